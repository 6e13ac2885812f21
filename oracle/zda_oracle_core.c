/*
 * ORACLE (test infrastructure, not product code).
 *
 * Plain float64 CPU leap-frog Yee update of one ZDA zone in cylindrical
 * coordinates (r, phi, z).  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may call this.  It shares
 * no code with the CUDA path under paper_2501_07979_b200/.
 *
 * What it follows:
 *   PAPER.md:53-62  Eq. 3-5  (reduced Maxwell equations, cylindrical curl D_m)
 *   PAPER.md:64     staggered Yee grid + leap-frog; r = 0 loop integral;
 *                   stretched-coordinate PML in r and z; Bloch-periodic phi
 *   SURVEY.md 8(c)  Steps 0-5 (the discrete reading of the above; readings
 *                   A1-A7, A10 are listed in DESIGN.md)
 *
 * Array layout here: C order, shape (Nr, Nphi, Nz), element [i][j][k],
 * k fastest.  (The CUDA library uses a different layout; nothing is shared.)
 *
 * Staggering (Step 0):
 *   Er  [i,j,k] @ (r_{i+1/2}, phi_j,       z_k      )
 *   Ephi[i,j,k] @ (r_i,       phi_{j+1/2}, z_k      )
 *   Ez  [i,j,k] @ (r_i,       phi_j,       z_{k+1/2})
 *   Hr  [i,j,k] @ (r_i,       phi_{j+1/2}, z_{k+1/2})
 *   Hphi[i,j,k] @ (r_{i+1/2}, phi_j,       z_{k+1/2})
 *   Hz  [i,j,k] @ (r_{i+1/2}, phi_{j+1/2}, z_k      )
 *
 * Built twice from this one source: real fields (symbols *_re) and complex
 * Bloch fields (-DZO_COMPLEX, symbols *_cx).  Compile with
 *   gcc -O2 -ffp-contract=off -fopenmp -fPIC -shared
 * No blocking, fusion or reordering beyond the update equations themselves;
 * OpenMP only splits the outermost (i) loop, whose iterations are independent.
 */
#include <complex.h>
#include <stddef.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#ifdef ZO_COMPLEX
typedef double complex T;
#define ZO_NAME(f) f##_cx
#define ZO_CONJ(x) conj(x)
#else
typedef double T;
#define ZO_NAME(f) f##_re
#define ZO_CONJ(x) (x)
#endif

/* Everything the update needs that is not a field.  All 1-D arrays are
 * computed by the Python side of the oracle (oracle/zone.py) in float64. */
typedef struct {
    int Nr, Nphi, Nz;
    int has_axis;            /* r_0 == 0: Step 5 */
    double dt, inv_dr, inv_dz;
    double phase_re, phase_im; /* p: F[., Nphi, .] = p F[., 0, .]  (Step 1) */
    /* per-r metric coefficients, length Nr (Eq. 5's 1/r factors) */
    const double *inv_rdphi_int;   /* 1/(r_i dphi); 0 on the axis            */
    const double *inv_rdphi_half;  /* 1/(r_{i+1/2} dphi)                     */
    const double *ca, *cb;         /* Hz: r_{i+1}/(r_{i+1/2}dr), r_i/(r_{i+1/2}dr) */
    const double *cc, *cd;         /* Ez: r_{i+1/2}/(r_i dr), r_{i-1/2}/(r_i dr)   */
    /* CPML b, c, 1/kappa (Step 2) at integer (_i) and half (_h) positions */
    const double *br_i, *cr_i, *ikr_i, *br_h, *cr_h, *ikr_h;   /* length Nr */
    const double *bz_i, *cz_i, *ikz_i, *bz_h, *cz_h, *ikz_h;   /* length Nz */
    /* Exact cylindrical PML ("r' = r + i zeta_r / omega ... regularised"; R25), rpml_exact != 0:
     * inside the OUTER r-slab (cells i >= Nr - npml_r_hi; the concave inner slab keeps the quasi form, where the exact one
     * is unstable) every 1/r factor becomes 1/r~, r~ = r + i zeta/omega,
     * realised as a second recursive-convolution operator Q[D] = D + chi, chi <- bq chi + cq D, with the coefficients of
     * sigma~ = zeta(r)/r and the regularising alpha~ > |sigma~| (length Nr, at integer and half positions);
     * hir_* = 1/(2 r) for the averaged F/r term of the radial derivative written in its split form. */
    int rpml_exact, npml_r_lo, npml_r_hi;
    const double *bq_i, *cq_i, *bq_h, *cq_h, *hir_i, *hir_h;
} zo_grid;

#ifndef ZO_COMPLEX
/* threads the i-loops below are split over (reported by bench.py's cpu_baseline) */
int zo_max_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
#endif

#define IDX(i, j, k) (((size_t)(i) * g->Nphi + (size_t)(j)) * g->Nz + (size_t)(k))

/* Step 2: the CPML operator P_a[D] = D/kappa + psi, psi <- b psi + c D first. */
static inline T cpml(T D, T *psi, double b, double c, double ik)
{
    *psi = b * (*psi) + c * D;
    return D * ik + (*psi);
}

/*
 * Step 3 -- H update (Faraday; Eq. 3 with the curl of Eq. 5):
 *   Hr   -= dt [ d+phi Ez /(r_i dphi)                    - Pz(d+z Ephi / dz) ]
 *   Hphi -= dt [ Pz(d+z Er / dz)                         - Pr(d+r Ez / dr)   ]
 *   Hz   -= dt [ Pr((r_{i+1}Ephi[i+1]-r_i Ephi[i])/(r_{i+1/2}dr)) - d+phi Er/(r_{i+1/2}dphi) ]
 * Ghosts (Step 1): E at i = Nr and k = Nz is 0; phi wraps with the phase p.
 * H-update CPML coefficients sit at the H component's own position: half in
 * z for Hr, Hphi; half in r for Hphi, Hz.
 */
void ZO_NAME(zo_update_H)(const zo_grid *g,
                          T *Hr, T *Hphi, T *Hz,
                          const T *Er, const T *Ephi, const T *Ez,
                          T *psi_Hr_z, T *psi_Hphi_z, T *psi_Hphi_r, T *psi_Hz_r,
                          T *chi_Hr, T *chi_Hz)
{
    const int Nr = g->Nr, Nphi = g->Nphi, Nz = g->Nz;
#ifdef ZO_COMPLEX
    const T p = g->phase_re + g->phase_im * I;
#else
    const T p = g->phase_re;
#endif
#pragma omp parallel for schedule(static)
    for (int i = 0; i < Nr; ++i) {
        for (int j = 0; j < Nphi; ++j) {
            const int jp = (j + 1 < Nphi) ? j + 1 : 0;
            const int wrap = (j + 1 == Nphi);
            for (int k = 0; k < Nz; ++k) {
                const size_t c = IDX(i, j, k);
                /* neighbours, with ghosts */
                const T Ez_jp   = wrap ? p * Ez[IDX(i, jp, k)] : Ez[IDX(i, jp, k)];
                const T Er_jp   = wrap ? p * Er[IDX(i, jp, k)] : Er[IDX(i, jp, k)];
                const T Ephi_kp = (k + 1 < Nz) ? Ephi[IDX(i, j, k + 1)] : 0.0;
                const T Er_kp   = (k + 1 < Nz) ? Er[IDX(i, j, k + 1)] : 0.0;
                const T Ez_ip   = (i + 1 < Nr) ? Ez[IDX(i + 1, j, k)] : 0.0;
                const T Ephi_ip = (i + 1 < Nr) ? Ephi[IDX(i + 1, j, k)] : 0.0;

                /* exact complex-r PML (R25): this cell lies in an r-slab */
                const int xr = g->rpml_exact && (i >= Nr - g->npml_r_hi);
                /* Hr (skipped on the axis, Step 5: r_0 = 0, held at 0) */
                if (!(g->has_axis && i == 0)) {
                    T t1 = (Ez_jp - Ez[c]) * g->inv_rdphi_int[i];
                    if (xr) t1 = cpml(t1, &chi_Hr[c], g->bq_i[i], g->cq_i[i], 1.0);     /* (1/r~) d_phi Ez */
                    const T Dz = (Ephi_kp - Ephi[c]) * g->inv_dz;
                    const T t2 = cpml(Dz, &psi_Hr_z[c], g->bz_h[k], g->cz_h[k], g->ikz_h[k]);
                    Hr[c] -= g->dt * (t1 - t2);
                }
                /* Hphi */
                {
                    const T Dz = (Er_kp - Er[c]) * g->inv_dz;
                    const T t1 = cpml(Dz, &psi_Hphi_z[c], g->bz_h[k], g->cz_h[k], g->ikz_h[k]);
                    const T Dr = (Ez_ip - Ez[c]) * g->inv_dr;
                    const T t2 = cpml(Dr, &psi_Hphi_r[c], g->br_h[i], g->cr_h[i], g->ikr_h[i]);
                    Hphi[c] -= g->dt * (t1 - t2);
                }
                /* Hz */
                if (!xr) {
                    const T Dr = Ephi_ip * g->ca[i] - Ephi[c] * g->cb[i];
                    const T t1 = cpml(Dr, &psi_Hz_r[c], g->br_h[i], g->cr_h[i], g->ikr_h[i]);
                    const T t2 = (Er_jp - Er[c]) * g->inv_rdphi_half[i];
                    Hz[c] -= g->dt * (t1 - t2);
                } else {
                    /* (1/(r~ s_r)) d_r(r~ Ephi) - (1/r~) d_phi Er = (1/s_r) d_r Ephi + (1/r~)[Ephi - d_phi Er], because
                     * d r~/dr = s_r; the conservative difference above IS (Ephi[i+1]-Ephi[i])/dr + (Ephi[i+1]+Ephi[i])/(2 r_{i+1/2}) */
                    const T Dr = (Ephi_ip - Ephi[c]) * g->inv_dr;
                    const T t1 = cpml(Dr, &psi_Hz_r[c], g->br_h[i], g->cr_h[i], g->ikr_h[i]);
                    const T q = (Ephi_ip + Ephi[c]) * g->hir_h[i] - (Er_jp - Er[c]) * g->inv_rdphi_half[i];
                    const T t2 = cpml(q, &chi_Hz[c], g->bq_h[i], g->cq_h[i], 1.0);
                    Hz[c] -= g->dt * (t1 + t2);
                }
            }
        }
    }
}

/*
 * Step 4 -- E update (Ampere; Eq. 4 with Eq. 5):
 *   Er   += (dt/eps) [ d-phi Hz /(r_{i+1/2}dphi)      - Pz(d-z Hphi / dz) - Jr   ]
 *   Ephi += (dt/eps) [ Pz(d-z Hr / dz)                - Pr(d-r Hz / dr)   - Jphi ]
 *   Ez   += (dt/eps) [ Pr((r_{i+1/2}Hphi[i]-r_{i-1/2}Hphi[i-1])/(r_i dr)) - d-phi Hr/(r_i dphi) ]
 * then the PEC zeros: Er, Ephi at k = 0; Ephi, Ez at i = 0 (annulus).
 * Step 5 (axis zone): Ephi[0] is skipped (held at 0); Ez[0,j,k] is one
 * unknown per k, replicated over j, from Ampere's law on the circle r = dr/2:
 *   Ez0[k] += (dt/eps0[k]) (4/dr) mean_j Hphi[0,j,k]        if p == 1,
 * held at 0 otherwise.  eps0[k] is the mean over j of eps[0,j,k] (DESIGN.md
 * reading R-axis-eps), passed in as cE_axis[k] = dt/eps0[k].
 * Step 6: J is non-zero only on plane k = source_k (r and phi components),
 * J_r / J_phi are (Nr, Nphi) planes for this step, or NULL.
 * cE[i,j,k] = dt/eps of the voxel (reading A3: one eps per voxel for its
 * three E components).
 */
void ZO_NAME(zo_update_E)(const zo_grid *g,
                          T *Er, T *Ephi, T *Ez,
                          const T *Hr, const T *Hphi, const T *Hz,
                          const double *cE, const double *cE_axis,
                          const T *J_r, const T *J_phi, int source_k,
                          T *psi_Er_z, T *psi_Ephi_z, T *psi_Ephi_r, T *psi_Ez_r,
                          T *chi_Er, T *chi_Ez)
{
    const int Nr = g->Nr, Nphi = g->Nphi, Nz = g->Nz;
#ifdef ZO_COMPLEX
    const T p = g->phase_re + g->phase_im * I;
#else
    const T p = g->phase_re;
#endif
    const T pbar = ZO_CONJ(p);
    const int p_is_one = (g->phase_re == 1.0 && g->phase_im == 0.0);
#pragma omp parallel for schedule(static)
    for (int i = 0; i < Nr; ++i) {
        for (int j = 0; j < Nphi; ++j) {
            const int jm = (j > 0) ? j - 1 : Nphi - 1;
            const int wrap = (j == 0);
            for (int k = 0; k < Nz; ++k) {
                const size_t c = IDX(i, j, k);
                const T Hz_jm   = wrap ? pbar * Hz[IDX(i, jm, k)] : Hz[IDX(i, jm, k)];
                const T Hr_jm   = wrap ? pbar * Hr[IDX(i, jm, k)] : Hr[IDX(i, jm, k)];
                const T Hphi_km = (k > 0) ? Hphi[IDX(i, j, k - 1)] : 0.0;
                const T Hr_km   = (k > 0) ? Hr[IDX(i, j, k - 1)] : 0.0;
                const T Hz_im   = (i > 0) ? Hz[IDX(i - 1, j, k)] : 0.0;
                const T Hphi_im = (i > 0) ? Hphi[IDX(i - 1, j, k)] : 0.0;
                const int on_src = (k == source_k);
                const T Jr   = (on_src && J_r)   ? J_r[(size_t)i * Nphi + j]   : 0.0;
                const T Jphi = (on_src && J_phi) ? J_phi[(size_t)i * Nphi + j] : 0.0;

                const int xr = g->rpml_exact && (i >= Nr - g->npml_r_hi);
                /* Er: PEC at k = 0 */
                if (k > 0) {
                    T t1 = (Hz[c] - Hz_jm) * g->inv_rdphi_half[i];
                    if (xr) t1 = cpml(t1, &chi_Er[c], g->bq_h[i], g->cq_h[i], 1.0);     /* (1/r~) d_phi Hz */
                    const T Dz = (Hphi[c] - Hphi_km) * g->inv_dz;
                    const T t2 = cpml(Dz, &psi_Er_z[c], g->bz_i[k], g->cz_i[k], g->ikz_i[k]);
                    Er[c] += cE[c] * (t1 - t2 - Jr);
                }
                /* Ephi: PEC at k = 0 and at i = 0 (wall, or the axis where it is held at 0) */
                if (k > 0 && i > 0) {
                    const T Dz = (Hr[c] - Hr_km) * g->inv_dz;
                    const T t1 = cpml(Dz, &psi_Ephi_z[c], g->bz_i[k], g->cz_i[k], g->ikz_i[k]);
                    const T Dr = (Hz[c] - Hz_im) * g->inv_dr;
                    const T t2 = cpml(Dr, &psi_Ephi_r[c], g->br_i[i], g->cr_i[i], g->ikr_i[i]);
                    Ephi[c] += cE[c] * (t1 - t2 - Jphi);
                }
                /* Ez: PEC at i = 0 for the annulus; axis handled below */
                if (i > 0 && !xr) {
                    const T Dr = Hphi[c] * g->cc[i] - Hphi_im * g->cd[i];
                    const T t1 = cpml(Dr, &psi_Ez_r[c], g->br_i[i], g->cr_i[i], g->ikr_i[i]);
                    const T t2 = (Hr[c] - Hr_jm) * g->inv_rdphi_int[i];
                    Ez[c] += cE[c] * (t1 - t2);
                } else if (i > 0) {
                    const T Dr = (Hphi[c] - Hphi_im) * g->inv_dr;
                    const T t1 = cpml(Dr, &psi_Ez_r[c], g->br_i[i], g->cr_i[i], g->ikr_i[i]);
                    const T q = (Hphi[c] + Hphi_im) * g->hir_i[i] - (Hr[c] - Hr_jm) * g->inv_rdphi_int[i];
                    const T t2 = cpml(q, &chi_Ez[c], g->bq_i[i], g->cq_i[i], 1.0);
                    Ez[c] += cE[c] * (t1 + t2);
                }
            }
        }
    }
    /* Step 5: the on-axis Ez (one unknown per k, replicated over j). */
    if (g->has_axis && p_is_one) {
        for (int k = 0; k < Nz; ++k) {
            T sum = 0.0;
            for (int j = 0; j < Nphi; ++j) sum += Hphi[IDX(0, j, k)];
            const T mean = sum / (double)Nphi;
            const T Ez0 = Ez[IDX(0, 0, k)] + cE_axis[k] * ((4.0 * g->inv_dr) * mean);
            for (int j = 0; j < Nphi; ++j) Ez[IDX(0, j, k)] = Ez0;
        }
    }
}
