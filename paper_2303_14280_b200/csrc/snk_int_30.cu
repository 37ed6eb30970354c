// integral-contraction kernel, class (l_a, l_b) = (3, 0)
#include "snk_int_kernel.cuh"
namespace snk { SNK_DEFINE_CLASS(3, 0) }
