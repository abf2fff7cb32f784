#include "dmx_inst.cuh"
DMX_INSTANTIATE(float, 1, ShapeDyn)
