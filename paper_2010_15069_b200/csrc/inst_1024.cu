// inst_1024.cu -- row/column pass kernels for line length 1024 (see launch.cuh)
#include "launch.cuh"
namespace spgpe {
SPGPE_DEFINE_LAUNCHERS(1024)
}
