#define TDH_NZ 32
#include "tile_inst.inc"
