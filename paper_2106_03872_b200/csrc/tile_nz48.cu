#define TDH_NZ 48
#include "tile_inst.inc"
