// fp32 instantiations of the right-hand-side column passes, run-time geometry (any grid and box; fwd_z of every plan): its own
// translation unit so that the build runs in parallel
#include "psfft_launch_impl.cuh"
namespace psfft { PSFFT_INSTANTIATE_COL(float, false) PSFFT_INSTANTIATE_FWDZ(float) }
