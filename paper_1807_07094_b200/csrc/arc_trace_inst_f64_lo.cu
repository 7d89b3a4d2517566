// arc_trace_inst_f64_lo.cu -- instantiates the tracer for double opacities, 1..4 frequency bins
#define ARC_INST_KT double
#define ARC_INST_NB0 1
#define ARC_INST_TAG f64_lo
#include "arc_trace_kernel.cuh"
