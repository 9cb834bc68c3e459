// qw_step_stream2d_f32.cu — complex64 instantiations of the streaming 2D kernel (qw_step_stream2d.cuh): the launcher and the
// general / Grover coins; the H (x) H and DFT coins are compiled in qw_step_stream2d_f32_b.cu (build time).
#include "qw_step_stream2d_host.cuh"

namespace qw {
QW_S2D_EXTERN(float, COIN_HXH4, false)
QW_S2D_EXTERN(float, COIN_DFT4, false)
int launch_stream2d_f32(qw_sim *s, int in_buf, int out_buf, int k, const Box &box) { return s2d_launch<float, false>(s, in_buf, out_buf, k, box); }
}  // namespace qw
