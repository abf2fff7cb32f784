#include "dmx_inst.cuh"
DMX_INSTANTIATE(double, 32, ShapeC4)
