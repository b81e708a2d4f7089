// psfft_f32_midx.cu -- float instantiations of the launchers, group MIDX (psfft_launch_impl.cuh).
#include "psfft_launch_impl.cuh"
namespace psfft {
PSFFT_INSTANTIATE_MIDX(float)
}
