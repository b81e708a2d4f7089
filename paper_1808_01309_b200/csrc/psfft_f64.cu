// psfft_f64.cu -- fp64 instantiations of the launchers.
#include "psfft_launch_impl.cuh"
namespace psfft {
PSFFT_INSTANTIATE(double)
}
