// qw_step_stream2d_rbl_f32.cu — complex64 instantiations of the streaming 2D kernel with random broken links drawn in the
// kernel (qw_step_stream2d.cuh, RBL = true; eqs. 9-10): the launcher and the
// general / Grover coins; the H (x) H and DFT coins are compiled in qw_step_stream2d_rbl_f32_b.cu (build time).
#include "qw_step_stream2d_host.cuh"

namespace qw {
QW_S2D_EXTERN(float, COIN_HXH4, true)
QW_S2D_EXTERN(float, COIN_DFT4, true)
int launch_stream2d_rbl_f32(qw_sim *s, int in_buf, int out_buf, int k, const Box &box) { return s2d_launch<float, true>(s, in_buf, out_buf, k, box); }
}  // namespace qw
