// libzda C ABI (include/zda.h): argument checks, the host-side grid/coefficient builder (a1),
// precision dispatch and the zone scheduler (a10).  Kernels live in zda_zone_impl.cuh.
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <exception>
#include <new>
#include "zda_common.h"

namespace zda {

static thread_local char g_err[1024] = "";

void set_error(const char* fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
}

int fail(int code, const char* fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
    return code;
}

static double cfl_limit_of(const zda_zone_desc& d) {
    // R10: dt <= 1/sqrt(1/dr^2 + 1/dz^2 + 1/(r_min dphi)^2), r_min = r_in (annulus) or dr/2 (axis)
    const double r_min = d.has_axis ? 0.5 * d.dr : d.r_in;
    const double a = r_min * d.dphi;
    double phi_term = 1.0 / (a * a);
    if (d.Nphi == 1) {
        // R21: with one phi cell the phi difference is the number (p - 1)/(r dphi); K = |p - 1|/dphi ~ |m|.
        // The 1/2 on the axis covers the 4/dr loop-integral update of Ez(0).
        const double K = std::hypot(d.phase_re - 1.0, d.phase_im) / d.dphi;
        phi_term = (K * K + (d.has_axis ? 0.5 : 0.0)) / (4.0 * r_min * r_min);
    }
    return 1.0 / std::sqrt(1.0 / (d.dr * d.dr) + 1.0 / (d.dz * d.dz) + phi_term);
}

int validate_desc(const zda_zone_desc* d, int max_steps) {
    if (!d) return fail(ZDA_E_BADARG, "desc is NULL");
    if (d->Nr < 2 || d->Nphi < 1 || d->Nz < 2) return fail(ZDA_E_BADARG, "grid %dx%dx%d too small", d->Nr, d->Nphi, d->Nz);
    if ((double)d->Nr * d->Nphi * d->Nz > 4.0e9) return fail(ZDA_E_BADARG, "grid too large");
    // launch-grid limits of the small kernels (gridDim.y = Nphi, gridDim.z = Nz / 2 or the design-layer thickness)
    if (d->Nphi > 65535) return fail(ZDA_E_BADARG, "Nphi = %d exceeds 65535", d->Nphi);
    if (d->Nz > 131070) return fail(ZDA_E_BADARG, "Nz = %d exceeds 131070", d->Nz);
    if (max_steps > (1 << 24)) return fail(ZDA_E_BADARG, "max_steps = %d exceeds %d", max_steps, 1 << 24);
    if (d->eps_volume != 0 && d->eps_volume != 1) return fail(ZDA_E_BADARG, "eps_volume must be 0 or 1");
    if (d->rpml_exact != 0 && d->rpml_exact != 1) return fail(ZDA_E_BADARG, "rpml_exact must be 0 or 1");
    if (d->rpml_exact) {
        // R25: the exact form grows slowly at small radius (x 10 over 32 000 steps at 200 cells, bounded from ~1000 on)
        if (d->npml_r_hi < 1) return fail(ZDA_E_BADARG, "rpml_exact needs an outer r-PML");
        const double r_slab = d->r_in + (d->Nr - d->npml_r_hi) * d->dr;
        if (r_slab < 1000.0 * d->dr)
            return fail(ZDA_E_BADARG, "rpml_exact: the outer r-slab starts at %.0f cells; the exact form is admitted from 1000 cells",
                        r_slab / d->dr);
    }
    if (!(d->dr > 0 && d->dz > 0 && d->dphi > 0 && d->dt > 0)) return fail(ZDA_E_BADARG, "dr, dphi, dz, dt must be > 0");
    if (d->n_fold < 0) return fail(ZDA_E_BADARG, "n_fold must be >= 0");
    if (d->n_fold > 0) {
        const double dphi_ref = 2.0 * M_PI / ((double)d->n_fold * d->Nphi);
        if (std::fabs(d->dphi - dphi_ref) > 1e-9 * dphi_ref) return fail(ZDA_E_BADARG, "dphi != 2 pi / (n_fold Nphi)");
    } else if (d->dphi * d->Nphi > 2.0 * M_PI * (1.0 + 1e-9)) {
        return fail(ZDA_E_BADARG, "wedge angle Nphi dphi exceeds 2 pi");
    }
    if (d->precision != 32 && d->precision != 64) return fail(ZDA_E_BADARG, "precision must be 32 or 64");
    if (d->has_axis) {
        if (d->r_in != 0.0) return fail(ZDA_E_BADARG, "has_axis needs r_in == 0");
        if (d->npml_r_lo != 0) return fail(ZDA_E_BADARG, "has_axis zone has no inner r-PML (PAPER.md:64)");
    } else if (!(d->r_in > 0)) {
        return fail(ZDA_E_BADARG, "annular zone needs r_in > 0");
    }
    const double pm = std::hypot(d->phase_re, d->phase_im);
    if (std::fabs(pm - 1.0) > 1e-9) return fail(ZDA_E_BADARG, "|phase| must be 1");
    if (!d->complex_fields && d->phase_im != 0.0) return fail(ZDA_E_BADARG, "real fields need a real phi-boundary phase");
    if (d->npml_r_lo < 0 || d->npml_r_hi < 0 || d->npml_z_lo < 0 || d->npml_z_hi < 0 ||
        d->npml_r_lo + d->npml_r_hi >= d->Nr || d->npml_z_lo + d->npml_z_hi >= d->Nz)
        return fail(ZDA_E_BADARG, "CPML slabs do not fit the grid");
    if (d->n_freq < 1 || d->n_freq > ZDA_MAX_FREQ || !d->omega) return fail(ZDA_E_BADARG, "n_freq must be 1..%d with omega set", ZDA_MAX_FREQ);
    // planes and the design box must sit outside the PMLs: the reciprocity the adjoint uses holds only there (R12)
    const int zlo = d->npml_z_lo, zhi = d->Nz - d->npml_z_hi;
    if (d->design_i0 < 0 || d->design_i1 > d->Nr || d->design_i0 >= d->design_i1) return fail(ZDA_E_BADARG, "design box r-range invalid");
    if (d->design_i0 < d->npml_r_lo || d->design_i1 > d->Nr - d->npml_r_hi) return fail(ZDA_E_BADARG, "design box inside the r-PML");
    if (d->design_k0 < zlo || d->design_k1 > zhi || d->design_k0 >= d->design_k1) return fail(ZDA_E_BADARG, "design box z-range invalid or inside the z-PML");
    if (d->monitor_k < zlo || d->monitor_k >= zhi) return fail(ZDA_E_BADARG, "monitor plane inside the z-PML");
    if (d->source_k < zlo || d->source_k >= zhi || d->source_k < 1) return fail(ZDA_E_BADARG, "source plane inside the z-PML");
    if (max_steps < 1) return fail(ZDA_E_BADARG, "max_steps must be >= 1");
    const double lim = cfl_limit_of(*d);
    if (d->dt > lim) return fail(ZDA_E_CFL, "dt = %.6g above the cylindrical CFL limit %.6g", d->dt, lim);
    return ZDA_OK;
}

// CFS-CPML tables along one axis (R5): depth x in [0,1] into a slab of npml cells,
// sigma = sigma_max x^p, kappa = 1 + (kappa_max - 1) x^p, alpha = alpha_max (1 - x),
// b = exp(-(sigma/kappa + alpha) dt), c = sigma (b - 1) / (sigma kappa + kappa^2 alpha).
static void cpml_axis(int N, int lo, int hi, const zda_zone_desc& d, double sigma_max, double off,
                      std::vector<double>& b, std::vector<double>& c, std::vector<double>& ik) {
    b.assign(N, 0.0);
    c.assign(N, 0.0);
    ik.assign(N, 1.0);
    for (int n = 0; n < N; ++n) {
        const double q = n + off;
        double x = 0.0;
        if (lo > 0 && q < lo) x = (lo - q) / lo;
        if (hi > 0 && q > N - hi) x = (q - (N - hi)) / hi;
        if (x <= 0.0) continue;
        const double xp = std::pow(x, d.cpml_p);
        const double sigma = sigma_max * xp;
        const double kappa = 1.0 + (d.cpml_kappa_max - 1.0) * xp;
        const double alpha = d.cpml_alpha_max * (1.0 - x);
        ik[n] = 1.0 / kappa;
        if (sigma > 0.0) {
            b[n] = std::exp(-(sigma / kappa + alpha) * d.dt);
            c[n] = sigma * (b[n] - 1.0) / (sigma * kappa + kappa * kappa * alpha);
        }
    }
}

void build_grid_tables(const zda_zone_desc& d, GridTables& g) {
    const int Nr = d.Nr, Nz = d.Nz;
    g.pitch = (Nr + 31) / 32 * 32;
    g.cfl_limit = cfl_limit_of(d);
    for (auto& v : g.rc) v.assign(Nr, 0.0);
    for (int i = 0; i < Nr; ++i) {
        // Eq. 5's 1/r factors at r_i and r_{i+1/2}, conservative radial differences (R1)
        const double ri = d.r_in + i * d.dr, rh = ri + 0.5 * d.dr, rm = ri - 0.5 * d.dr;
        g.rc[RC_INV_RDPHI_HALF][i] = 1.0 / (rh * d.dphi);
        g.rc[RC_CA][i] = (ri + d.dr) / (rh * d.dr);
        g.rc[RC_CB][i] = ri / (rh * d.dr);
        if (ri > 0.0) {
            g.rc[RC_INV_RDPHI_INT][i] = 1.0 / (ri * d.dphi);
            g.rc[RC_CC][i] = rh / (ri * d.dr);
            g.rc[RC_CD][i] = rm / (ri * d.dr);
        }
        // weights of the objective / gradient (R9): the radius of each component's own position
        g.rc[RC_W_HALF][i] = rh;
        g.rc[RC_W_INT][i] = ri;
        g.rc[RC_W_Z][i] = (d.has_axis && i == 0) ? d.dr / 8.0 : ri;
    }
    cpml_axis(Nr, d.npml_r_lo, d.npml_r_hi, d, d.cpml_sigma_max_r, 0.0, g.rc[RC_B_I], g.rc[RC_C_I], g.rc[RC_IK_I]);
    cpml_axis(Nr, d.npml_r_lo, d.npml_r_hi, d, d.cpml_sigma_max_r, 0.5, g.rc[RC_B_H], g.rc[RC_C_H], g.rc[RC_IK_H]);
    // R25: the 1/r~ operator of the exact outer r-PML: sigma~ = zeta / r with zeta the integral of sigma from the slab's
    // interface, alpha~ the slab's own CFS shift; hir = 1 / (2 r)
    for (int h = 0; h < 2; ++h) {
        const double off = h ? 0.5 : 0.0;
        std::vector<double>&bq = g.rc[h ? RC_BQ_H : RC_BQ_I], &cq = g.rc[h ? RC_CQ_H : RC_CQ_I], &hir = g.rc[h ? RC_HIR_H : RC_HIR_I];
        for (int i = 0; i < Nr; ++i) {
            const double q = i + off, r = d.r_in + q * d.dr;
            hir[i] = r > 0.0 ? 1.0 / (2.0 * r) : 0.0;
            if (d.npml_r_hi < 1 || !(q > Nr - d.npml_r_hi)) continue;
            const double x = (q - (Nr - d.npml_r_hi)) / d.npml_r_hi;
            const double zeta = d.cpml_sigma_max_r * (d.npml_r_hi * d.dr) * std::pow(x, d.cpml_p + 1.0) / (d.cpml_p + 1.0);
            const double sig = zeta / r, alpha = d.cpml_alpha_max * (1.0 - x);
            if (sig > 0.0) {
                bq[i] = std::exp(-(sig + alpha) * d.dt);
                cq[i] = sig * (bq[i] - 1.0) / (sig + alpha);
            }
        }
    }
    for (auto& v : g.zc) v.assign(Nz, 0.0);
    cpml_axis(Nz, d.npml_z_lo, d.npml_z_hi, d, d.cpml_sigma_max_z, 0.0, g.zc[ZC_B_I], g.zc[ZC_C_I], g.zc[ZC_IK_I]);
    cpml_axis(Nz, d.npml_z_lo, d.npml_z_hi, d, d.cpml_sigma_max_z, 0.5, g.zc[ZC_B_H], g.zc[ZC_C_H], g.zc[ZC_IK_H]);
}

// Gauss-Jordan with partial pivoting, in place.
bool invert_real(std::vector<double>& a, int n) {
    std::vector<double> inv(n * n, 0.0);
    for (int i = 0; i < n; ++i) inv[i * n + i] = 1.0;
    for (int col = 0; col < n; ++col) {
        int piv = col;
        for (int r = col + 1; r < n; ++r)
            if (std::fabs(a[r * n + col]) > std::fabs(a[piv * n + col])) piv = r;
        if (a[piv * n + col] == 0.0) return false;
        if (piv != col)
            for (int c = 0; c < n; ++c) {
                std::swap(a[piv * n + c], a[col * n + c]);
                std::swap(inv[piv * n + c], inv[col * n + c]);
            }
        const double s = 1.0 / a[col * n + col];
        for (int c = 0; c < n; ++c) { a[col * n + c] *= s; inv[col * n + c] *= s; }
        for (int r = 0; r < n; ++r) {
            if (r == col) continue;
            const double f = a[r * n + col];
            if (f == 0.0) continue;
            for (int c = 0; c < n; ++c) { a[r * n + c] -= f * a[col * n + c]; inv[r * n + c] -= f * inv[col * n + c]; }
        }
    }
    a = inv;
    return true;
}

// complex n x n inverse through the real 2n x 2n embedding [[Re, -Im], [Im, Re]]
bool invert_complex(std::vector<double>& a_re, std::vector<double>& a_im, int n) {
    const int m = 2 * n;
    std::vector<double> big(m * m);
    for (int r = 0; r < n; ++r)
        for (int c = 0; c < n; ++c) {
            big[r * m + c] = a_re[r * n + c];
            big[r * m + (c + n)] = -a_im[r * n + c];
            big[(r + n) * m + c] = a_im[r * n + c];
            big[(r + n) * m + (c + n)] = a_re[r * n + c];
        }
    if (!invert_real(big, m)) return false;
    for (int r = 0; r < n; ++r)
        for (int c = 0; c < n; ++c) {
            a_re[r * n + c] = big[r * m + c];
            a_im[r * n + c] = big[(r + n) * m + c];
        }
    return true;
}

}  // namespace zda

using namespace zda;

// Nothing throws across the ABI: every entry point that can reach an allocation or a container runs its body under
// this guard (std::bad_alloc -> ZDA_E_NOMEM, any other exception -> ZDA_E_BADARG with its text).
#define ZDA_TRY try {
#define ZDA_CATCH                                                                                           \
    } catch (const std::bad_alloc&) {                                                                       \
        return fail(ZDA_E_NOMEM, "out of host memory (std::bad_alloc) in %s", __func__);                    \
    } catch (const std::exception& e) {                                                                     \
        return fail(ZDA_E_BADARG, "%s: exception: %s", __func__, e.what());                                 \
    } catch (...) {                                                                                         \
        return fail(ZDA_E_BADARG, "%s: unknown exception", __func__);                                       \
    }

extern "C" {

const char* zda_last_error(void) { return g_err; }

size_t zda_zone_workspace_bytes(const zda_zone_desc* desc, int max_steps) {
    try {
        if (validate_desc(desc, max_steps) != ZDA_OK) return 0;
        return desc->precision == 64 ? workspace_bytes_f64(*desc, max_steps) : workspace_bytes_f32(*desc, max_steps);
    } catch (...) {
        fail(ZDA_E_NOMEM, "exception in zda_zone_workspace_bytes");
        return 0;
    }
}

int zda_zone_create(const zda_zone_desc* desc, const double* eps_bg_z, int max_steps, void* workspace,
                    size_t bytes, void* stream, zda_zone** out) {
    ZDA_TRY
    if (!out) return fail(ZDA_E_BADARG, "out is NULL");
    *out = nullptr;
    int rc = validate_desc(desc, max_steps);
    if (rc != ZDA_OK) return rc;
    if (!workspace) return fail(ZDA_E_BADARG, "workspace is NULL");
    if ((reinterpret_cast<uintptr_t>(workspace) & 255u) != 0) return fail(ZDA_E_BADARG, "workspace must be 256-byte aligned");
    if (eps_bg_z)
        for (int k = 0; k < desc->Nz; ++k)
            if (!(eps_bg_z[k] > 0)) return fail(ZDA_E_BADARG, "eps_bg_z[%d] must be > 0", k);
    ZoneBase* impl = nullptr;
    rc = desc->precision == 64
             ? create_zone_f64(*desc, eps_bg_z, max_steps, workspace, bytes, (cudaStream_t)stream, &impl)
             : create_zone_f32(*desc, eps_bg_z, max_steps, workspace, bytes, (cudaStream_t)stream, &impl);
    if (rc != ZDA_OK) return rc;
    zda_zone* handle = new (std::nothrow) zda_zone{impl};
    if (!handle) { delete impl; return fail(ZDA_E_NOMEM, "out of host memory"); }
    *out = handle;
    return ZDA_OK;
    ZDA_CATCH
}

int zda_zone_destroy(zda_zone* z) {
    ZDA_TRY
    if (!z) return ZDA_OK;
    delete z->impl;
    delete z;
    return ZDA_OK;
    ZDA_CATCH
}

#define ZDA_NEED(z) if (!(z) || !(z)->impl) return fail(ZDA_E_BADARG, "zone is NULL")

int zda_set_option(zda_zone* z, int option, int value) {
    ZDA_TRY
    ZDA_NEED(z);
    return z->impl->set_option(option, value);
    ZDA_CATCH
}

int zda_set_design_eps(zda_zone* z, const void* eps_design, int on_host) {
    ZDA_TRY
    ZDA_NEED(z);
    if (!eps_design) return fail(ZDA_E_BADARG, "eps_design is NULL");
    return z->impl->set_design_eps(eps_design, on_host);
    ZDA_CATCH
}

int zda_set_eps_volume(zda_zone* z, const void* eps, int on_host) {
    ZDA_TRY
    ZDA_NEED(z);
    if (!eps) return fail(ZDA_E_BADARG, "eps is NULL");
    return z->impl->set_eps_volume(eps, on_host);
    ZDA_CATCH
}

int zda_set_density(zda_zone* z, const void* rho2d, int on_host, double eps0, double eps_h,
                    double filt_sigma, double beta, double eta) {
    ZDA_TRY
    ZDA_NEED(z);
    if (!rho2d) return fail(ZDA_E_BADARG, "rho2d is NULL");
    if (!(eps0 > 0 && eps_h > 0)) return fail(ZDA_E_BADARG, "eps0, eps_h must be > 0");
    if (!(filt_sigma > 0) || std::ceil(3.0 * filt_sigma) > 48) return fail(ZDA_E_BADARG, "filt_sigma must be in (0, 16]");
    if (!(beta > 0) || !(eta > 0 && eta < 1)) return fail(ZDA_E_BADARG, "need beta > 0 and 0 < eta < 1");
    return z->impl->set_density(rho2d, on_host, 0, eps0, eps_h, filt_sigma, beta, eta);
    ZDA_CATCH
}

int zda_set_density_conic(zda_zone* z, const void* rho2d, int on_host, double eps0, double eps_h,
                          double radius, double beta, double eta) {
    ZDA_TRY
    ZDA_NEED(z);
    if (!rho2d) return fail(ZDA_E_BADARG, "rho2d is NULL");
    if (!(eps0 > 0 && eps_h > 0)) return fail(ZDA_E_BADARG, "eps0, eps_h must be > 0");
    if (!(radius > 0)) return fail(ZDA_E_BADARG, "conic radius must be > 0");
    if (!(beta > 0) || !(eta > 0 && eta < 1)) return fail(ZDA_E_BADARG, "need beta > 0 and 0 < eta < 1");
    return z->impl->set_density(rho2d, on_host, 1, eps0, eps_h, radius, beta, eta);
    ZDA_CATCH
}

int zda_set_source(zda_zone* z, int n_terms, const void* A_r, const void* A_phi, int on_host,
                   const double* s_table, int Nt) {
    ZDA_TRY
    ZDA_NEED(z);
    if (n_terms < 1 || n_terms > ZDA_MAX_TERMS) return fail(ZDA_E_BADARG, "n_terms must be 1..%d", ZDA_MAX_TERMS);
    if (!A_r || !A_phi || !s_table || Nt < 1) return fail(ZDA_E_BADARG, "source arrays missing");
    return z->impl->set_source(n_terms, A_r, A_phi, on_host, s_table, Nt);
    ZDA_CATCH
}

int zda_run_forward(zda_zone* z, int n_steps) {
    ZDA_TRY
    ZDA_NEED(z);
    if (n_steps < 0) return fail(ZDA_E_BADARG, "n_steps < 0");
    return z->impl->run_forward(n_steps);
    ZDA_CATCH
}

int zda_set_focal_weights(zda_zone* z, const void* g, const double* u, int on_host) {
    ZDA_TRY
    ZDA_NEED(z);
    if (!g) return fail(ZDA_E_BADARG, "zda_set_focal_weights: g is NULL");
    return z->impl->set_focal_weights(g, u, on_host);
    ZDA_CATCH
}

int zda_build_focal_weights(zda_zone* z, double focal_dz, const double* u) {
    ZDA_TRY
    ZDA_NEED(z);
    if (!(focal_dz > 0)) return fail(ZDA_E_BADARG, "zda_build_focal_weights: focal_dz must be > 0");
    return z->impl->build_focal_weights(focal_dz, u);
    ZDA_CATCH
}

int zda_get_focal_sums(zda_zone* z, double* S) {
    ZDA_TRY
    ZDA_NEED(z);
    if (!S) return fail(ZDA_E_BADARG, "zda_get_focal_sums: S is NULL");
    return z->impl->get_focal_sums(S);
    ZDA_CATCH
}

int zda_build_adjoint_source(zda_zone* z, int objective, double t0, double sigma_t, int n_steps, double* F_out) {
    ZDA_TRY
    ZDA_NEED(z);
    if (objective != ZDA_OBJ_MONITOR_ENERGY && objective != ZDA_OBJ_FOCAL_INTENSITY)
        return fail(ZDA_E_BADARG, "unknown objective %d", objective);
    if (!(sigma_t > 0) || n_steps < 1) return fail(ZDA_E_BADARG, "need sigma_t > 0 and n_steps >= 1");
    return z->impl->build_adjoint_source(objective, t0, sigma_t, n_steps, F_out);
    ZDA_CATCH
}

int zda_run_adjoint(zda_zone* z, int n_steps) {
    ZDA_TRY
    ZDA_NEED(z);
    if (n_steps < 0) return fail(ZDA_E_BADARG, "n_steps < 0");
    return z->impl->run_adjoint(n_steps);
    ZDA_CATCH
}

int zda_pair_run_forward(zda_zone* a, zda_zone* b, int n_steps) {
    ZDA_TRY
    ZDA_NEED(a);
    ZDA_NEED(b);
    if (n_steps < 0) return fail(ZDA_E_BADARG, "n_steps < 0");
    return a->impl->run_batch(b->impl, ZDA_FWD, n_steps);
    ZDA_CATCH
}

int zda_pair_run_adjoint(zda_zone* a, zda_zone* b, int n_steps) {
    ZDA_TRY
    ZDA_NEED(a);
    ZDA_NEED(b);
    if (n_steps < 0) return fail(ZDA_E_BADARG, "n_steps < 0");
    return a->impl->run_batch(b->impl, ZDA_ADJ, n_steps);
    ZDA_CATCH
}

// While zones on DIFFERENT streams are in flight together, a persistent cooperative kernel (ZDA_KERNEL_PERSIST under AUTO)
// would hold every SM for its whole run; the schedulers tell the zones so (measured: config8 40 -> 36 Gvox/s otherwise).
struct ConcurrentHint {
    zda_zone** zones; int n; bool on = false;
    ConcurrentHint(zda_zone** z, int n_) : zones(z), n(n_) {
        for (int l = 1; l < n; ++l) if (zones[l]->impl->stream() != zones[0]->impl->stream()) on = true;
        if (on) for (int l = 0; l < n; ++l) zones[l]->impl->hint_concurrent(true);
    }
    ~ConcurrentHint() { if (on) for (int l = 0; l < n; ++l) zones[l]->impl->hint_concurrent(false); }
};

// Scheduler helper: run `which` on zones l and l + 1 in shared launches when they can be batched (NEXT-4), else on zone l
// alone; returns the number of zones it ran (1 or 2) or a negative error code.
static int run_one_or_pair(zda_zone** zones, int n_zones, int l, int which, const int* n_steps) {
    zda::ZoneBase* z = zones[l]->impl;
    if (l + 1 < n_zones && n_steps[l] == n_steps[l + 1] && z->can_batch_with(zones[l + 1]->impl)) {
        int rc = z->run_batch(zones[l + 1]->impl, which, n_steps[l]);
        return rc != ZDA_OK ? rc : 2;
    }
    int rc = which == ZDA_FWD ? z->run_forward(n_steps[l]) : z->run_adjoint(n_steps[l]);
    return rc != ZDA_OK ? rc : 1;
}

int zda_get_dft(zda_zone* z, int which, int region, int comp, int freq, void* out, int on_host) {
    ZDA_TRY
    ZDA_NEED(z);
    if (!out) return fail(ZDA_E_BADARG, "out is NULL");
    return z->impl->get_dft(which, region, comp, freq, out, on_host);
    ZDA_CATCH
}

int zda_get_field(zda_zone* z, int comp, void* out, int on_host) {
    ZDA_TRY
    ZDA_NEED(z);
    if (!out) return fail(ZDA_E_BADARG, "out is NULL");
    if (comp < ZDA_ER || comp > ZDA_HZ) return fail(ZDA_E_BADARG, "comp out of range");
    return z->impl->get_field(comp, out, on_host);
    ZDA_CATCH
}

int zda_gradient(zda_zone* z, void* dF_deps, void* dF_deps_zsum, void* dF_drho, int on_host) {
    ZDA_TRY
    ZDA_NEED(z);
    return z->impl->gradient(dF_deps, dF_deps_zsum, dF_drho, on_host);
    ZDA_CATCH
}

int zda_check_finite(zda_zone* z) {
    ZDA_TRY
    ZDA_NEED(z);
    return z->impl->check_finite();
    ZDA_CATCH
}

int zda_schedule_bytes(zda_zone* z, int which, double* out) {
    ZDA_TRY
    ZDA_NEED(z);
    if (!out || (which != ZDA_FWD && which != ZDA_ADJ)) return fail(ZDA_E_BADARG, "zda_schedule_bytes: bad argument");
    return z->impl->schedule_bytes(which, out);
    ZDA_CATCH
}

long long zda_launch_count(const zda_zone* z) { return (z && z->impl) ? z->impl->launch_count() : 0; }

const char* zda_kernel_name(const zda_zone* z) { return (z && z->impl) ? z->impl->kernel_name() : ""; }

// a10: zones are independent units; one GPU runs them.  The zones are driven phase by phase (all forward
// runs enqueued, then every adjoint source, then all adjoint runs, then the gradients): members on DIFFERENT streams
// then overlap on the GPU, which is what fills the machine when a zone is smaller than one wave of CTAs (the paper's thin
// wedges and its first zone).  Zones on one stream run back to back.
int zda_lens_gradient(zda_zone** zones, int n_zones, const int* n_steps_fwd, const int* n_steps_adj,
                      const double* adj_t0, const double* adj_sigma_t, double* F_out,
                      void** dF_deps_zsum, void** dF_drho) {
    ZDA_TRY
    if (!zones || n_zones < 1 || !n_steps_fwd || !n_steps_adj || !adj_t0 || !adj_sigma_t)
        return fail(ZDA_E_BADARG, "zda_lens_gradient: missing argument");
    for (int l = 0; l < n_zones; ++l) { ZDA_NEED(zones[l]); }
    ConcurrentHint concurrent(zones, n_zones);
    // Resident zones cannot share workspace memory: creation and the zda_set_* calls have already written each zone's
    // tables, materials and sheets into its workspace.  (One buffer reused down a list of zones means creating, solving
    // and destroying them one at a time, as bench.py's config5 does.)
    for (int l = 0; l < n_zones; ++l) {
        const char *alo, *ahi, *blo, *bhi;
        zones[l]->impl->workspace_range(&alo, &ahi);
        for (int a = 0; a < l; ++a) {
            zones[a]->impl->workspace_range(&blo, &bhi);
            if (!(ahi <= blo || bhi <= alo)) return fail(ZDA_E_BADARG, "zones %d and %d share workspace memory", a, l);
        }
    }
    {
        const int g0 = 0, g1 = n_zones;
        for (int l = g0; l < g1; ++l) {
            int rc = zones[l]->impl->run_forward(n_steps_fwd[l]);
            if (rc != ZDA_OK) return rc;
        }
        for (int l = g0; l < g1; ++l) {          // synchronises zone l's stream only
            zda::ZoneBase* z = zones[l]->impl;
            const int objective = z->has_focal_weights() ? ZDA_OBJ_FOCAL_INTENSITY : ZDA_OBJ_MONITOR_ENERGY;
            double F = 0.0;
            int rc = z->build_adjoint_source(objective, adj_t0[l], adj_sigma_t[l], n_steps_adj[l], &F);
            if (rc != ZDA_OK) return rc;
            if (F_out) F_out[l] = F;
            rc = z->run_adjoint(n_steps_adj[l]);   // enqueued at once, so this zone keeps the GPU busy while the next waits
            if (rc != ZDA_OK) return rc;
        }
        for (int l = g0; l < g1; ++l) {
            void* gz = dF_deps_zsum ? dF_deps_zsum[l] : nullptr;
            void* gr = dF_drho ? dF_drho[l] : nullptr;
            if (gz || gr) {
                int rc = zones[l]->impl->gradient(nullptr, gz, gr, 0);
                if (rc != ZDA_OK) return rc;
            }
        }
    }
    return ZDA_OK;
    ZDA_CATCH
}

// The paper's lens objective: the zones -- and the m = +1 / m = -1 members of a pair -- add
// coherently at the focal point.  Same phase-by-phase schedule as zda_lens_gradient; the one extra step is the sum of
// the zones' S_f between the forward and the adjoint phase.
int zda_lens_focal_gradient(zda_zone** zones, int n_zones, const int* n_steps_fwd, const int* n_steps_adj,
                            const double* adj_t0, const double* adj_sigma_t, const double* u, double* F_out,
                            double* S_out, void** dF_deps_zsum, void** dF_drho) {
    ZDA_TRY
    if (!zones || n_zones < 1 || !n_steps_fwd || !n_steps_adj || !adj_t0 || !adj_sigma_t)
        return fail(ZDA_E_BADARG, "zda_lens_focal_gradient: missing argument");
    for (int l = 0; l < n_zones; ++l) { ZDA_NEED(zones[l]); }
    ConcurrentHint concurrent(zones, n_zones);
    const int F = zones[0]->impl->n_freq();
    for (int l = 0; l < n_zones; ++l) {
        if (zones[l]->impl->n_freq() != F) return fail(ZDA_E_BADARG, "zone %d has a different n_freq", l);
        if (!zones[l]->impl->has_focal_weights()) return fail(ZDA_E_STATE, "zone %d has no focal weights", l);
        const char *alo, *ahi, *blo, *bhi;
        zones[l]->impl->workspace_range(&alo, &ahi);
        for (int a = 0; a < l; ++a) {      // every zone's forward DFT must survive until the sum is known
            zones[a]->impl->workspace_range(&blo, &bhi);
            if (!(ahi <= blo || bhi <= alo)) return fail(ZDA_E_BADARG, "zones %d and %d share workspace memory", a, l);
        }
    }
    for (int l = 0; l < n_zones;) {
        int ran = run_one_or_pair(zones, n_zones, l, ZDA_FWD, n_steps_fwd);
        if (ran < 0) return ran;
        l += ran;
    }
    double S[2 * ZDA_MAX_FREQ] = {0.0};
    for (int l = 0; l < n_zones; ++l) {
        double Sl[2 * ZDA_MAX_FREQ];
        int rc = zones[l]->impl->get_focal_sums(Sl);
        if (rc != ZDA_OK) return rc;
        for (int t = 0; t < 2 * F; ++t) S[t] += Sl[t];
    }
    double Ftot = 0.0;
    for (int f = 0; f < F; ++f) Ftot += (u ? u[f] : 1.0) * (S[2 * f] * S[2 * f] + S[2 * f + 1] * S[2 * f + 1]);
    if (F_out) *F_out = Ftot;
    if (S_out) for (int t = 0; t < 2 * F; ++t) S_out[t] = S[t];
    for (int l = 0; l < n_zones; ++l) {
        int rc = zones[l]->impl->build_adjoint_source(ZDA_OBJ_FOCAL_INTENSITY, adj_t0[l], adj_sigma_t[l], n_steps_adj[l],
                                                      nullptr, S, u);
        if (rc != ZDA_OK) return rc;
    }
    for (int l = 0; l < n_zones;) {
        int ran = run_one_or_pair(zones, n_zones, l, ZDA_ADJ, n_steps_adj);
        if (ran < 0) return ran;
        l += ran;
    }
    for (int l = 0; l < n_zones; ++l) {
        void* gz = dF_deps_zsum ? dF_deps_zsum[l] : nullptr;
        void* gr = dF_drho ? dF_drho[l] : nullptr;
        if (gz || gr) {
            int rc = zones[l]->impl->gradient(nullptr, gz, gr, 0);
            if (rc != ZDA_OK) return rc;
        }
    }
    return ZDA_OK;
    ZDA_CATCH
}

}  // extern "C"
