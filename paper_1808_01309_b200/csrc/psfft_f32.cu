// psfft_f32.cu -- fp32 instantiations of the launchers.
#include "psfft_launch_impl.cuh"
namespace psfft {
PSFFT_INSTANTIATE(float)
}
