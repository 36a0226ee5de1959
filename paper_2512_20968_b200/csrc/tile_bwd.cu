// tile_bwd.cu -- mesh_attn_tile_bwd (placeholder until the tcgen05 backward kernel lands)
#include "tile_kernels.hpp"
namespace mesh_attn {
int launch_tile_bwd(const BwdParams&, const CUtensorMap&, const CUtensorMap&, const CUtensorMap&, const CUtensorMap&, int, cudaStream_t)
{
    return (int)cudaErrorNotSupported;
}
}  // namespace mesh_attn
