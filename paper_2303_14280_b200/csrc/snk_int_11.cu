// integral-contraction kernel, class (l_a, l_b) = (1, 1)
#include "snk_int_kernel.cuh"
namespace snk { SNK_DEFINE_CLASS(1, 1) }
