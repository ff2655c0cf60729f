#define TDH_NZ 64
#include "tile_inst.inc"
