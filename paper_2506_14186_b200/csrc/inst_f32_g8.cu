#include "dmx_inst.cuh"
DMX_INSTANTIATE(float, 8, ShapeDyn)
