// qw_step_stream2d_rbl_f32_b.cu — second half of qw_step_stream2d_rbl_f32.cu: the H (x) H and DFT coin instances (build time).
#include "qw_step_stream2d_host.cuh"

namespace qw {
QW_S2D_DEFINE(float, COIN_HXH4, true)
QW_S2D_DEFINE(float, COIN_DFT4, true)
}  // namespace qw
