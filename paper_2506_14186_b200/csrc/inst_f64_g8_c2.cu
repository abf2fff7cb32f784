#include "dmx_inst.cuh"
DMX_INSTANTIATE(double, 8, ShapeC2)
