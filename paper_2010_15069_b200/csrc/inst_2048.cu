// inst_2048.cu -- row/column pass kernels for line length 2048 (see launch.cuh)
#include "launch.cuh"
namespace spgpe {
SPGPE_DEFINE_LAUNCHERS(2048)
}
