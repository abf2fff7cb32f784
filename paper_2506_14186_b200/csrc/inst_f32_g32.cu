#include "dmx_inst.cuh"
DMX_INSTANTIATE(float, 32, ShapeDyn)
