#include "dmx_inst.cuh"
DMX_INSTANTIATE(double, 16, ShapeC3)
