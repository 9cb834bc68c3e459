// qw_step_stream2d_f32_b.cu — second half of qw_step_stream2d_f32.cu: the H (x) H and DFT coin instances (build time).
#include "qw_step_stream2d_host.cuh"

namespace qw {
QW_S2D_DEFINE(float, COIN_HXH4, false)
QW_S2D_DEFINE(float, COIN_DFT4, false)
}  // namespace qw
