// psfft_f32_col.cu -- float instantiations of the launchers, group COL (psfft_launch_impl.cuh).
#include "psfft_launch_impl.cuh"
namespace psfft {
PSFFT_INSTANTIATE_COL(float)
}
