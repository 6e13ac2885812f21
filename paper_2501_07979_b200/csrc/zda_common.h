// Internal host-side declarations of libzda (not part of the ABI).
#pragma once
#include <cuda_runtime.h>
#include <cstddef>
#include <cstdint>
#include <string>
#include <vector>
#include "../../include/zda.h"

namespace zda {

// thread-local error text behind zda_last_error()
void set_error(const char* fmt, ...);
int fail(int code, const char* fmt, ...);

#define ZDA_CUDA_OK(expr)                                                                     \
    do {                                                                                      \
        cudaError_t e__ = (expr);                                                             \
        if (e__ != cudaSuccess)                                                               \
            return ::zda::fail(ZDA_E_CUDA, "%s failed: %s (%s:%d)", #expr, cudaGetErrorString(e__), \
                               __FILE__, __LINE__);                                           \
    } while (0)

// Bump allocator over the caller's workspace; with base == nullptr it only measures.
struct Arena {
    char* base = nullptr;
    size_t off = 0;
    template <class P> P* take(size_t count) {
        off = (off + 255) & ~size_t(255);
        P* p = base ? reinterpret_cast<P*>(base + off) : nullptr;
        off += count * sizeof(P);
        return p;
    }
};

// a1: everything the grid builder derives from the description, in double (host).
enum { RC_INV_RDPHI_INT = 0, RC_INV_RDPHI_HALF, RC_CA, RC_CB, RC_CC, RC_CD,
       RC_B_I, RC_C_I, RC_IK_I, RC_B_H, RC_C_H, RC_IK_H, RC_W_HALF, RC_W_INT, RC_W_Z,
       RC_BQ_I, RC_CQ_I, RC_BQ_H, RC_CQ_H, RC_HIR_I, RC_HIR_H,      // R25: the 1/r~ operator of the exact outer r-PML
       RC_COUNT };
enum { ZC_B_I = 0, ZC_C_I, ZC_IK_I, ZC_B_H, ZC_C_H, ZC_IK_H, ZC_CE_BG, ZC_CE_AXIS, ZC_COUNT };
struct GridTables {
    int pitch = 0;                       // row pitch in elements (multiple of 32)
    std::vector<double> rc[RC_COUNT];    // per-r tables, length Nr (see the enum)
    std::vector<double> zc[ZC_COUNT];    // per-z tables, length Nz (CE_* filled by the zone)
    double cfl_limit = 0;
};

// Ghost rows on each side of phi in the field layout: 2 where the two-step kernel (two-row halo) can run, else 1.
inline int field_ghost(const zda_zone_desc& d) { return (d.Nphi >= 16 && !d.has_axis) ? 2 : 1; }

int validate_desc(const zda_zone_desc* d, int max_steps);
void build_grid_tables(const zda_zone_desc& d, GridTables& g);

// Precision-independent interface; one implementation per Real in zda_zone_impl.cuh.
struct ZoneBase {
    virtual ~ZoneBase() {}
    virtual int set_option(int option, int value) = 0;
    virtual int set_design_eps(const void* eps, int on_host) = 0;
    virtual int set_eps_volume(const void* eps, int on_host) = 0;
    virtual int set_density(const void* rho, int on_host, int filter_mode, double eps0, double eps_h, double width,
                            double beta, double eta) = 0;
    virtual int set_source(int n_terms, const void* A_r, const void* A_phi, int on_host,
                           const double* s_table, int Nt) = 0;
    virtual int set_focal_weights(const void* g, const double* u, int on_host) = 0;
    virtual int build_focal_weights(double focal_dz, const double* u) = 0;
    virtual bool has_focal_weights() const = 0;
    virtual int n_freq() const = 0;
    virtual int get_focal_sums(double* S) = 0;
    virtual int run_forward(int n_steps) = 0;
    // S_total (focal intensity only, may be NULL): 2 n_freq doubles (re, im), the coherent focal field to use in place of
    // the zone's own S_f, with weights u_total (n_freq, NULL = ones) in place of the zone's
    virtual int build_adjoint_source(int objective, double t0, double sigma_t, int n_steps, double* F_out,
                                     const double* S_total = nullptr, const double* u_total = nullptr) = 0;
    virtual int run_adjoint(int n_steps) = 0;
    // NEXT-4: both zones advance in the same launches (one-step fused kernel); which = ZDA_FWD | ZDA_ADJ
    virtual bool can_batch_with(ZoneBase* other) const = 0;
    virtual int run_batch(ZoneBase* other, int which, int n_steps) = 0;
    virtual int get_dft(int which, int region, int comp, int freq, void* out, int on_host) = 0;
    virtual int get_field(int comp, void* out, int on_host) = 0;
    virtual int gradient(void* dF_deps, void* dF_deps_zsum, void* dF_drho, int on_host) = 0;
    virtual int check_finite() = 0;
    // scheduler hint: other zones run on other streams at the same time (a persistent kernel would hold every SM)
    virtual int hint_concurrent(bool on) = 0;
    virtual int schedule_bytes(int which, double* out) = 0;
    virtual long long launch_count() const = 0;
    virtual const char* kernel_name() const = 0;
    virtual cudaStream_t stream() const = 0;
    virtual void workspace_range(const char** lo, const char** hi) const = 0;
};

size_t workspace_bytes_f32(const zda_zone_desc& d, int max_steps);
size_t workspace_bytes_f64(const zda_zone_desc& d, int max_steps);
int create_zone_f32(const zda_zone_desc& d, const double* eps_bg_z, int max_steps, void* ws, size_t bytes,
                    cudaStream_t stream, ZoneBase** out);
int create_zone_f64(const zda_zone_desc& d, const double* eps_bg_z, int max_steps, void* ws, size_t bytes,
                    cudaStream_t stream, ZoneBase** out);

// small dense solves for the adjoint-source builder (host, double)
bool invert_real(std::vector<double>& a, int n);                        // in place, row-major n x n
bool invert_complex(std::vector<double>& a_re, std::vector<double>& a_im, int n);

}  // namespace zda

struct zda_zone {
    zda::ZoneBase* impl;
};
