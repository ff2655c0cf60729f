#define TDH_NZ 48
#include "plane_inst.inc"
