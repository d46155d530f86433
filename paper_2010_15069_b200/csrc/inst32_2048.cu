// inst32_2048.cu -- fp32 row/column pass kernels for line length 2048 (see launch32.cuh)
#include "launch32.cuh"
namespace spgpe {
SPGPE_DEFINE_LAUNCHERS32(2048)
}
