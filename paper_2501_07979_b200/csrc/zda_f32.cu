// fp32 instantiation of the zone (the product precision).
#include "zda_zone_impl.cuh"
namespace zda {
size_t workspace_bytes_f32(const zda_zone_desc& d, int max_steps) { return workspace_bytes_impl<float>(d, max_steps); }
int create_zone_f32(const zda_zone_desc& d, const double* eps_bg_z, int max_steps, void* ws, size_t bytes,
                    cudaStream_t stream, ZoneBase** out) {
    return create_zone_impl<float>(d, eps_bg_z, max_steps, ws, bytes, stream, out);
}
}  // namespace zda
