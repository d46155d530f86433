// inst_256.cu -- row/column pass kernels for line length 256 (see launch.cuh)
#include "launch.cuh"
namespace spgpe {
SPGPE_DEFINE_LAUNCHERS(256)
}
