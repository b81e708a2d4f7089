// fp64 instantiations of the right-hand-side column passes, compile-time geometry (N^3 grid, 2 pi box): its own
// translation unit so that the build runs in parallel
#include "psfft_launch_impl.cuh"
namespace psfft { PSFFT_INSTANTIATE_COL(double, true) }
