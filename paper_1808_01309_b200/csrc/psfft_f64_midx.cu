// psfft_f64_midx.cu -- double instantiations of the launchers, group MIDX (psfft_launch_impl.cuh).
#include "psfft_launch_impl.cuh"
namespace psfft {
PSFFT_INSTANTIATE_MIDX(double)
}
