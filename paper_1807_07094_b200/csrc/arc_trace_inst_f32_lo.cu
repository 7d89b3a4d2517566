// arc_trace_inst_f32_lo.cu -- instantiates the tracer for float opacities, 1..4 frequency bins
#define ARC_INST_KT float
#define ARC_INST_NB0 1
#define ARC_INST_TAG f32_lo
#include "arc_trace_kernel.cuh"
