#define TDH_NZ 16
#include "plane_inst.inc"
