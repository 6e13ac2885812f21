// fp64 instantiation of the zone (parity build): this translation unit is compiled with
// -fmad=false so that every expression is evaluated exactly in the order it is written.
#include "zda_zone_impl.cuh"
namespace zda {
size_t workspace_bytes_f64(const zda_zone_desc& d, int max_steps) { return workspace_bytes_impl<double>(d, max_steps); }
int create_zone_f64(const zda_zone_desc& d, const double* eps_bg_z, int max_steps, void* ws, size_t bytes,
                    cudaStream_t stream, ZoneBase** out) {
    return create_zone_impl<double>(d, eps_bg_z, max_steps, ws, bytes, stream, out);
}
}  // namespace zda
