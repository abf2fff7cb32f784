#include "dmx_inst.cuh"
DMX_INSTANTIATE(double, 1, ShapeDyn)
