#define TDH_NZ 64
#include "plane_inst.inc"
