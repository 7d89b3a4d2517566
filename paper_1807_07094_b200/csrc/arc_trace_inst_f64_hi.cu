// arc_trace_inst_f64_hi.cu -- instantiates the tracer for double opacities, 5..8 frequency bins
#define ARC_INST_KT double
#define ARC_INST_NB0 5
#define ARC_INST_TAG f64_hi
#include "arc_trace_kernel.cuh"
