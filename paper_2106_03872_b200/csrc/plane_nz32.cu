#define TDH_NZ 32
#include "plane_inst.inc"
