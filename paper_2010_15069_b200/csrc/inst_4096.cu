// inst_4096.cu -- row/column pass kernels for line length 4096 (see launch.cuh)
#include "launch.cuh"
namespace spgpe {
SPGPE_DEFINE_LAUNCHERS(4096)
}
