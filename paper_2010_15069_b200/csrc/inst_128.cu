// inst_128.cu -- row/column pass kernels for line length 128 (see launch.cuh)
#include "launch.cuh"
namespace spgpe {
SPGPE_DEFINE_LAUNCHERS(128)
}
