// inst_512.cu -- row/column pass kernels for line length 512 (see launch.cuh)
#include "launch.cuh"
namespace spgpe {
SPGPE_DEFINE_LAUNCHERS(512)
}
