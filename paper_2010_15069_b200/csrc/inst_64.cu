// inst_64.cu -- row/column pass kernels for line length 64 (see launch.cuh)
#include "launch.cuh"
namespace spgpe {
SPGPE_DEFINE_LAUNCHERS(64)
}
