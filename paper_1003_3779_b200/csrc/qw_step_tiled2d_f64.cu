// qw_step_tiled2d_f64.cu — complex128 instantiations of the register-tiled 2D kernel (qw_step_tiled2d.cuh).
#include "qw_step_tiled2d_host.cuh"

namespace qw {
int launch_tiled2d_f64(qw_sim *s, int in_buf, int out_buf, int k, const Box &box) { return t2d_launch<double>(s, in_buf, out_buf, k, box); }
}  // namespace qw
