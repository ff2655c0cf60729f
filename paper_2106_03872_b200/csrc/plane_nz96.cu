#define TDH_NZ 96
#include "plane_inst.inc"
