// inst32_4096.cu -- fp32 row/column pass kernels for line length 4096 (see launch32.cuh)
#include "launch32.cuh"
namespace spgpe {
SPGPE_DEFINE_LAUNCHERS32(4096)
}
