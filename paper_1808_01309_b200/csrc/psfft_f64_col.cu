// psfft_f64_col.cu -- double instantiations of the launchers, group COL (psfft_launch_impl.cuh).
#include "psfft_launch_impl.cuh"
namespace psfft {
PSFFT_INSTANTIATE_COL(double)
}
