#define TDH_NZ 16
#include "tile_inst.inc"
