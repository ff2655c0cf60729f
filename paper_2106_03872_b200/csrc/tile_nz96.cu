#define TDH_NZ 96
#include "tile_inst.inc"
