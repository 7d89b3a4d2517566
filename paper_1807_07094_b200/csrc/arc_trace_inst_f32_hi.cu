// arc_trace_inst_f32_hi.cu -- instantiates the tracer for float opacities, 5..8 frequency bins
#define ARC_INST_KT float
#define ARC_INST_NB0 5
#define ARC_INST_TAG f32_hi
#include "arc_trace_kernel.cuh"
