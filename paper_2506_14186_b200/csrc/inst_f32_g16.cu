#include "dmx_inst.cuh"
DMX_INSTANTIATE(float, 16, ShapeDyn)
