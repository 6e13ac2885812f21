/*
 * zda.h -- C ABI of libzda: the differentiable cylindrical-coordinate FDTD solve of one
 * ZDA (zoned discrete axisymmetry) zone on one B200 (sm_100a).
 *
 * Method: arxiv 2501.07979.  The zone problem is PAPER.md:33-62 (Eq. 1-5: the
 * Bloch-periodic wedge and the reduced Maxwell equations with the cylindrical curl D_m),
 * its discretisation PAPER.md:64 (staggered Yee grid, leap-frog, r = 0 loop integral,
 * stretched-coordinate PML in r and z), the running DTFT and the hybrid time/frequency
 * adjoint PAPER.md:66-68, the density map Eq. 6 PAPER.md:72-76 and the filters :83.
 * The discrete reading of all of this is DESIGN.md ("Readings" R1-R23).
 *
 * Conventions
 *   - every call returns int: ZDA_OK (0) or a negative ZDA_E_* code; zda_last_error()
 *     gives a thread-local text for the last failure.  Nothing throws or aborts across
 *     the ABI: every entry point catches C++ exceptions (std::bad_alloc -> ZDA_E_NOMEM, any
 *     other -> ZDA_E_BADARG).  A failed call leaves the zone usable unless the code is ZDA_E_CUDA.
 *   - units: c = eps_0 = mu_0 = 1, mu = 1; e^{-i omega t} time convention.
 *   - cells (i, j, k), 0 <= i < Nr, 0 <= j < Nphi, 0 <= k < Nz; boxes are half-open.
 *   - ARRAY LAYOUT at this boundary: dense, r fastest:  a[(k*Nphi + j)*Nr + i]
 *     ("[k][j][i]"); plane arrays a[j*Nr + i]; box arrays use the box extents in the
 *     same order.  Element type is float (precision == 32) or double (precision == 64);
 *     complex elements are interleaved (re, im) pairs of that type.  Field arrays are
 *     complex iff desc.complex_fields; DFT arrays are always complex.
 *   - `on_host` arguments say where a caller array lives: 0 = device memory of the
 *     current CUDA device (e.g. torch.Tensor.data_ptr()), 1 = host memory (pinned or
 *     pageable).  Arguments documented as "host" are always host pointers.
 *   - ownership: the caller owns every buffer it passes, including the workspace, which
 *     must stay alive and untouched until zda_zone_destroy.  The library allocates no
 *     device memory of its own (PyTorch is the only allocator); it copies what it needs
 *     into the workspace.
 *   - all device work is enqueued on the `stream` given at creation (a cudaStream_t passed
 *     as void*; NULL = the legacy default stream).  Calls that return values to the host
 *     (F_out, on_host outputs) synchronise that stream before returning; all others are
 *     asynchronous.
 *   - not thread-safe per zone; different zones may be driven from different threads.
 */
#ifndef ZDA_H_
#define ZDA_H_

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

/* every entry point below is exported from libzda.so (the rest of the library is hidden) */
#if defined(__GNUC__)
#define ZDA_API __attribute__((visibility("default")))
#else
#define ZDA_API
#endif

#define ZDA_OK          0
#define ZDA_E_BADARG   (-1)  /* NULL pointer, size/box out of range, plane inside a PML ... */
#define ZDA_E_CFL      (-2)  /* dt above the cylindrical CFL limit (R10)                    */
#define ZDA_E_NOMEM    (-3)  /* workspace too small, or out of host memory                  */
#define ZDA_E_CUDA     (-4)  /* a CUDA runtime/driver call failed (text has the error)      */
#define ZDA_E_STATE    (-5)  /* call order: e.g. run_adjoint before build_adjoint_source    */
#define ZDA_E_NAN      (-6)  /* non-finite field: zda_check_finite, or a run with ZDA_OPT_CHECK_EVERY */

/* field components (zda_get_field, zda_get_dft) */
enum { ZDA_ER = 0, ZDA_EPHI = 1, ZDA_EZ = 2, ZDA_HR = 3, ZDA_HPHI = 4, ZDA_HZ = 5 };
/* which run / which region (zda_get_dft) */
enum { ZDA_FWD = 0, ZDA_ADJ = 1 };
enum { ZDA_DESIGN = 0, ZDA_MONITOR = 1 };
/* objective (zda_build_adjoint_source) */
enum { ZDA_OBJ_MONITOR_ENERGY = 0,    /* F = sum W |Ehat(monitor)|^2 (R9)                                   */
       ZDA_OBJ_FOCAL_INTENSITY = 1 }; /* F = sum_f u_f |S_f|^2, needs zda_set_focal_weights (Eq. 7; R20)   */
/* time-loop kernel selection (zda_set_option ZDA_OPT_KERNEL) */
enum { ZDA_KERNEL_AUTO = 0,      /* FUSED2 where it applies, else FUSED where it applies, else PERSIST / SPLIT */
       ZDA_KERNEL_SPLIT = 1,     /* two passes per step: H-update kernel, E-update kernel       */
       ZDA_KERNEL_FUSED = 2,     /* one pass per step: TMA-tiled fused H+E kernel (no axis)     */
       ZDA_KERNEL_FUSED2 = 3,    /* one pass per TWO steps: temporally blocked TMA-tiled kernel; needs Nphi >= 16, no axis,
                                    no rpml_exact; AUTO takes it wherever it applies */
       ZDA_KERNEL_PERSIST = 4 }; /* small zones: ONE persistent cooperative kernel steps the whole run (grid barriers
                                    between the H and E passes, state resident in L2); every zone type, incl. axis zones;
                                    ZDA_E_BADARG if the zone's state exceeds 96 MB.  AUTO takes it for axis zones that fit */
enum { ZDA_OPT_KERNEL = 0,       /* one of ZDA_KERNEL_*                                         */
       ZDA_OPT_ADJ_MONITOR_DFT = 1, /* 1: the adjoint run also accumulates the monitor plane (default 0) */
       /* Tuning knobs of the fused kernel's launch plan; 0 = the plan's own choice.  Results do not
          depend on them (tests/test_gpu_knobs.py runs the fp64 parity under every value).                        */
       ZDA_OPT_FUSED_TJ = 2,      /* tile rows per CTA: 6 | 7 (one-step kernel), 5 | 9 | 13 (two-step kernel) */
       ZDA_OPT_FUSED_CHUNK = 3,   /* planes per z-chunk                                          */
       ZDA_OPT_FUSED_CLUSTER = 4, /* phi-neighbouring tiles per thread-block cluster, 1..8       */
       ZDA_OPT_DFT_PERIOD = 5,    /* steps between visits of the design-box accumulators: 2 | 4 | 8, at most the period
                                     the workspace's ring was sized for at creation (else ZDA_E_BADARG)            */
       ZDA_OPT_SPLIT_GRAPH = 6,   /* 0: the split path uses plain launches instead of a CUDA graph (default 1)     */
       /* Failure detector inside the runs: after every K-th step E is scanned for non-finite values; the
          run call then synchronises and returns ZDA_E_NAN at once (a CFL / PML blow-up does not burn the rest of the
          horizon).  0 = off (default; runs are then fully asynchronous).                                          */
       ZDA_OPT_CHECK_EVERY = 7 };

/*
 * One zone (Fig. 2 :51): the annular wedge r_in <= r < r_in + Nr dr,
 * 0 <= phi < 2 pi / n_fold, 0 <= z < Nz dz, with dphi = 2 pi / (n_fold Nphi).
 * Staggering (R1): Er @ (i+1/2, j, k), Ephi @ (i, j+1/2, k), Ez @ (i, j, k+1/2),
 * Hr @ (i, j+1/2, k+1/2), Hphi @ (i+1/2, j, k+1/2), Hz @ (i+1/2, j+1/2, k); E at t = n dt,
 * H at (n+1/2) dt.  PEC box behind the PMLs (R7).
 */
typedef struct zda_zone_desc {
    int    Nr, Nphi, Nz;
    double dr, dphi, dz;        /* dphi must equal 2 pi / (n_fold Nphi) to 1e-9 relative when
                                   n_fold > 0                                                  */
    double r_in;                /* inner radius; 0 iff has_axis                                */
    double dt;                  /* <= 1/sqrt(1/dr^2 + 1/dz^2 + 1/(r_min dphi)^2), r_min = r_in
                                   (annulus) or dr/2 (axis); else ZDA_E_CFL (R10).  With Nphi == 1
                                   (the continuously axisymmetric first zone; R21) the
                                   phi term is (K^2 + 1/2 [axis]) / (2 r_min)^2, K = |p - 1| / dphi */
    int    n_fold;              /* n_i of PAPER.md:33; 0 = a wedge of angle Nphi dphi that is not
                                   an integer fraction of the circle (cut-down test zones)      */
    double phase_re, phase_im;  /* phi-boundary phase p: F[., Nphi, .] = p F[., 0, .] (Eq. 1-2,
                                   PAPER.md:37-47; R2).  |p| must be 1.                         */
    int    complex_fields;      /* 0: real fields (p must be +-1); 1: complex (Bloch) fields   */
    int    has_axis;            /* r_in == 0: loop-integral axis (R4), then
                                   npml_r_lo must be 0                                          */
    /* CFS-CPML ("stretched-coordinate PMLs"; R5, R6): slab thickness in cells and the
       polynomial profile sigma = sigma_max x^p, kappa = 1 + (kappa_max-1) x^p, alpha = alpha_max (1-x) */
    int    npml_r_lo, npml_r_hi, npml_z_lo, npml_z_hi;
    double cpml_p, cpml_sigma_max_r, cpml_sigma_max_z, cpml_kappa_max, cpml_alpha_max;
    /* design box [design_i0, design_i1) x all j x [design_k0, design_k1): per-voxel eps and DFT     */
    int    design_i0, design_i1, design_k0, design_k1;
    int    monitor_k;           /* DFT monitor plane (objective, adjoint source); outside z-PML */
    int    source_k;            /* forward current sheet plane; outside z-PML                  */
    int    n_freq;              /* number of design frequencies, 1..ZDA_MAX_FREQ               */
    const double* omega;        /* host, n_freq angular frequencies                            */
    int    precision;           /* 32: float kernels.  64: double kernels built with -fmad=false */
    int    rpml_exact;          /* 1: exact cylindrical PML in the OUTER r-slab (complex radius
                                   r~ = r + i zeta_r/omega; R25): every 1/r factor there becomes 1/r~ through a
                                   second recursive-convolution operator (4 more auxiliaries in that slab); reflection 30-40
                                   times below the quasi-CPML's (1.5e-5 at r = 1100 cells, 12 cells thick).  The concave inner
                                   slab keeps the quasi form (the exact one is unstable there), and the outer slab must start
                                   at a radius of at least 1000 dr (below that the exact form grows slowly: ZDA_E_BADARG).
                                   Kernels: ZDA_KERNEL_SPLIT and ZDA_KERNEL_FUSED.  0: quasi-CPML in both slabs (R6). */
    int    eps_volume;          /* 1: the workspace holds a per-voxel dt/eps for EVERY plane (4 or 8 bytes per voxel
                                   more) and zda_set_eps_volume may be called; 0: eps(z) + the design box only      */
} zda_zone_desc;
/* Limits (ZDA_E_BADARG beyond them): Nr * Nphi * Nz <= 4e9, Nphi <= 65535, Nz <= 131070, max_steps <= 2^24.
 * The quasi-CPML in r (R6) reflects about 1e-2 where the r-PML sits at radii below ~100 cells; R6. */

#define ZDA_MAX_FREQ  8
#define ZDA_MAX_TERMS 16   /* upper bound of source terms per sheet; a zone holds max(2, n_freq) terms with complex
                              fields and max(2, 2 n_freq) with real fields (zda_set_source: ZDA_E_BADARG beyond) */

typedef struct zda_zone zda_zone;   /* opaque; host memory owned by the library */

/* Text of the last failure on this thread ("" if none).  Never NULL. */
ZDA_API const char* zda_last_error(void);

/* Bytes of device workspace zda_zone_create needs for this description (0 on a bad
 * description; zda_last_error says why).  Covers fields (double-buffered), CPML
 * auxiliaries (slabs only), per-voxel dt/eps on the design box, 1-D coefficient tables,
 * DFT accumulators of both runs, source sheets and tables for up to `max_steps` steps, and -- where the
 * accumulators are visited every 4th or 8th step (several frequencies) -- a ring of 2 or 6 design-layer
 * copies of E. */
ZDA_API size_t zda_zone_workspace_bytes(const zda_zone_desc* desc, int max_steps);

/* a1: build the grid: per-r curl coefficients (Eq. 5's 1/r factors),
 * CPML tables, CFL check; carve the workspace; zero all state.  eps_bg_z: host, Nz doubles,
 * the 1-D background permittivity eps(z) (NULL = vacuum).  workspace: device, >= 256-byte
 * aligned, `bytes` >= zda_zone_workspace_bytes(desc, max_steps). */
ZDA_API int zda_zone_create(const zda_zone_desc* desc, const double* eps_bg_z, int max_steps,
                    void* workspace, size_t bytes, void* stream, zda_zone** out);

ZDA_API int zda_zone_destroy(zda_zone* z);

ZDA_API int zda_set_option(zda_zone* z, int option, int value);

/* Per-voxel permittivity on the design box (R3: one eps per voxel for its three E components):
 * eps_design[(kd*Nphi + j)*Nr_d + id], real, precision of the zone. */
ZDA_API int zda_set_design_eps(zda_zone* z, const void* eps_design, int on_host);

/* Per-voxel permittivity over the WHOLE zone (north_star "zda_zone_create with ... per-voxel eps"; a patterned
 * substrate, a second patterned layer): eps[(k*Nphi + j)*Nr + i] > 0, real, precision of the zone; replaces eps(z)
 * everywhere.  Needs desc.eps_volume = 1 (else ZDA_E_STATE).  A later zda_set_design_eps / zda_set_density overwrites
 * the design box only.  On an axis zone the on-axis Ez uses the phi-mean of eps[k][.][0] (R4). */
ZDA_API int zda_set_eps_volume(zda_zone* z, const void* eps, int on_host);

/* a2: density -> eps on the device (Eq. 6; filter/projection :83, R13, R14):
 * rho2d[j*Nr_d + id] in [0,1] -> separable Gaussian filter (sigma cells, truncated at
 * ceil(3 sigma), r edge-clamped, phi periodic) -> tanh projection (beta, eta) ->
 * eps = eps0 + rho_bar (eps_h - eps0), extruded over the design layer.  The parameters are
 * remembered for the VJP in zda_gradient. */
ZDA_API int zda_set_density(zda_zone* z, const void* rho2d, int on_host, double eps0, double eps_h,
                    double filt_sigma, double beta, double eta);

/* The same map with the paper's conic filter (PAPER.md:87 "a conic filter with a radius of 0.08 lambda", :133
 * "0.056 lambda"; R22) in place of the Gaussian: design cell (id, j) has its centre at
 * r = r_in + (design_i0 + id + 1/2) dr; the distance to cell (id', j + b) is d = sqrt(((id - id') dr)^2 + (rbar b dphi)^2)
 * with rbar the mean of the two radii; w = max(0, 1 - d / radius); b runs over all periodic images (cell (j + b) mod
 * Nphi); the sum is truncated at the design region's r edges; rho_f = sum w rho / sum w.  radius in the units of dr.
 * ZDA_E_BADARG if the cone reaches more than 4096 phi cells at the inner design radius. */
ZDA_API int zda_set_density_conic(zda_zone* z, const void* rho2d, int on_host, double eps0, double eps_h,
                          double radius, double beta, double eta);

/* a5: forward current sheet on plane source_k ("normally-incident plane wave"; R15):
 * J_c^{n+1/2}(i,j) = sum_q A_c[q][j][i] * s_table[q][n], c in {r, phi}.  A_*: n_terms planes,
 * field element type.  s_table: host doubles, n_terms x Nt (x2 interleaved re,im if
 * complex_fields), sampled by the caller at t = (n + 1/2) dt; J = 0 for n >= Nt. */
ZDA_API int zda_set_source(zda_zone* z, int n_terms, const void* A_r, const void* A_phi, int on_host,
                   const double* s_table, int Nt);

/* a3-a6: reset all state, then n_steps leap-frog steps (H-update, E-update, source, running DFT
 * Ehat_{c,f} += dt exp(+i omega_f (n+1) dt) E_c^{n+1} on the design box and the monitor plane;
 * PAPER.md:64, :68; R8).  Asynchronous. */
ZDA_API int zda_run_forward(zda_zone* z, int n_steps);

/* a7: objective F = sum_f sum_{c in r,phi} sum_{i outside r-PML, j} W_c(i) |Ehat^fwd_{c,f}(i,j,k_m)|^2
 * (R9) and the broadband adjoint source (R11): basis pulses
 * q_f(t) = exp(-(t-t0)^2 / 2 sigma_t^2) exp(-i omega_f (t-t0)) and per-point coefficients beta such that
 * the half-step DTFT of the adjoint current at every omega_f' equals conj(Ehat^fwd_{c,f'}(i,j,k_m)).
 * n_steps = length of the adjoint run the pulses are sampled for.  F_out: host, may be NULL. */
ZDA_API int zda_build_adjoint_source(zda_zone* z, int objective, double t0, double sigma_t, int n_steps,
                             double* F_out);

/* Focal-intensity objective (Eq. 7; R20): F = sum_f u_f |S_f|^2 with
 * S_f = sum_{c in r,phi} sum_{i outside r-PML, j} g[f][c][j][i] * Ehat^fwd_{c,f}(i, j, monitor_k), the field at the focal
 * point as a linear functional of the monitor-plane field.  g: the caller's near-to-far weights, n_freq x 2 x Nphi x Nr
 * complex elements of the zone's precision (host or device per on_host); u: host, n_freq doubles, NULL = all ones.
 * zda_build_adjoint_source(ZDA_OBJ_FOCAL_INTENSITY) then prescribes a_{c,f} = u_f conj(S_f) g_{c,f} / W_c.
 * The weights are copied into the workspace (into the adjoint run's monitor accumulators, so they cannot be combined with
 * ZDA_OPT_ADJ_MONITOR_DFT: ZDA_E_STATE) and stay set for every later run of the zone. */
ZDA_API int zda_set_focal_weights(zda_zone* z, const void* g, const double* u, int on_host);

/* The same objective with the weights BUILT by the library's near-to-far transform (Eq. 7-8: the focal
 * intensity of the x-polarised plane wave; R24): the half-space above the monitor plane is homogeneous with
 * eps_bg_z[monitor_k], so the x component of the field at the ON-AXIS point focal_dz above the plane is the first
 * Rayleigh-Sommerfeld integral of the plane's tangential field,
 *     S_f = -(1 / 2 pi) Int E_x(r') d/dz [exp(i k_f R) / R] dS',  k_f = omega_f sqrt(eps),  R = sqrt(rho'^2 + focal_dz^2),
 * with E_x = E_r cos(phi) - E_phi sin(phi) at each component's Yee position, dS = r dr dphi there, the zone's annulus
 * outside its r-PML as the aperture, and the other n_fold - 1 wedges of the circle entering through the Bloch
 * continuation (cos(phi) -> sum_w p^w cos(phi + w tau); non-zero only for m = +-1 mod n_fold: PAPER.md:76).
 * Replaces zda_set_focal_weights' g; u as there.  focal_dz > 0 in the units of dr. */
ZDA_API int zda_build_focal_weights(zda_zone* z, double focal_dz, const double* u);

/* S_f of the last forward run for every design frequency: S[2 f] = Re S_f, S[2 f + 1] = Im S_f (host, 2 n_freq doubles).
 * The per-frequency focal intensities I(p, omega_f) = |S_f|^2 are the constraint values of the epigraph form
 * (Eq. 7-8); its multipliers go back in as u.  Synchronises. */
ZDA_API int zda_get_focal_sums(zda_zone* z, double* S);

/* a8: adjoint run ("2 FDTD runs"): state reset, conjugate phi-phase (R12), the
 * source of zda_build_adjoint_source on plane monitor_k, DFT on the design box.  Asynchronous. */
ZDA_API int zda_run_adjoint(zda_zone* z, int n_steps);

/* NEXT-4 (the x-polarised plane wave is the sum of its m = +1 and m = -1 components, two zone problems on ONE
 * structure): zones a and b advance TOGETHER, one kernel launch per time step for both (the member comes from the block
 * index; each brings its own fields, CPML state, accumulators, sheets and phase).  Same semantics and results as
 * zda_run_forward / zda_run_adjoint on each of them (bit-identical), but a thin wedge that fills half a wave of CTAs alone
 * then fills the machine.  Requirements (else ZDA_E_BADARG with the reason): both zones run the one-step fused kernel
 * with the same launch plan, have the same grid, CPML, design box, n_freq and precision, sit on the same stream and in
 * separate workspaces; the adjoint call needs zda_build_adjoint_source on both (ZDA_E_STATE).  zda_lens_focal_gradient
 * batches consecutive zones that qualify by itself. */
ZDA_API int zda_pair_run_forward(zda_zone* a, zda_zone* b, int n_steps);
ZDA_API int zda_pair_run_adjoint(zda_zone* a, zda_zone* b, int n_steps);

/* Ehat_{comp,freq} of run `which` on `region`: design box [kd][j][id] or monitor plane [j][i],
 * complex, precision of the zone. */
ZDA_API int zda_get_dft(zda_zone* z, int which, int region, int comp, int freq, void* out, int on_host);

/* Current time-domain field component (ZDA_ER..ZDA_HZ), [k][j][i], field element type. */
ZDA_API int zda_get_field(zda_zone* z, int comp, void* out, int on_host);

/* a9: dF/deps(i,j,k) = sum_f sum_c 2 Re[(-i Omega_f) W_c(i) Ehat^fwd_{c,f} Ehat^adj_{c,f}],
 * Omega_f = (2/dt) sin(omega_f dt / 2) (north_star; R9-R12), on the design box.
 * Outputs (each may be NULL), real, precision of the zone:
 *   dF_deps       design box [kd][j][id]
 *   dF_deps_zsum  [j][id], summed over the layer in ascending kd (R19; one thread per (id, j) walks the layer, so the
 *                 sum stays in a register: with r fastest in memory there is nothing for a warp shuffle to reduce)
 *   dF_drho       [j][id], the VJP of zda_set_density (needs a prior zda_set_density) */
ZDA_API int zda_gradient(zda_zone* z, void* dF_deps, void* dF_deps_zsum, void* dF_drho, int on_host);

/* The dF_drho tail of zda_gradient as a stand-alone call that ALLOCATES NOTHING, for callers that cannot call
 * cudaMalloc or carve a workspace (code under CUDA graph capture, tight serving loops, harnesses that forbid it):
 * dF_drho = filter^T [ dF_deps_zsum (eps_h - eps0) d rho_bar / d rho_f ], rho_f = filter(rho2d), the Gaussian filter and
 * tanh projection of zda_set_density (Eq. 6; R13, R14) -- the same kernels, in the same order, as
 * zda_gradient runs them.  No zone handle: the caller passes the inputs and the output.
 *   precision      32 | 64: element type of the three arrays (float | double)
 *   rho2d, dF_deps_zsum (inputs), dF_drho (output): DEVICE pointers, dense [Nphi][Nr_d]; dF_drho may not alias an input
 *   stream         a cudaStream_t (NULL = the default stream); the call enqueues five kernels and returns, no sync
 * Scratch: the two intermediate planes sit in a static __device__ array of ZDA_STATIC_SCRATCH_BYTES that is part of
 * libzda.so -- every GPU that loads the library holds these 16 MiB until the process exits.  Limit: 2 planes of
 * Nr_d * Nphi elements, each rounded up to 256 B, must fit: at most 2 Mi cells in fp32, 1 Mi in fp64; beyond that the call
 * returns ZDA_E_BADARG (text names the sizes) and launches nothing -- use zda_gradient, whose scratch is the caller's.
 * Every call on a device shares the array, which keeps the last call's contents.  Nothing in it has to start at zero
 * (each kernel reads only what an earlier kernel of the same call wrote), so there is no clearing step; but two calls
 * that OVERLAP on the GPU (different streams, or different host threads on different streams) RACE on it: keep calls on
 * one stream, or order them with events.  The first call on each device looks the array's device address up
 * (cudaGetSymbolAddress, with that device current): make that first call outside a graph capture.
 * No cudaMalloc, cudaFree, or allocating library routine is called, and no host heap is used. */
#define ZDA_STATIC_SCRATCH_BYTES (16u << 20)
ZDA_API int zda_density_vjp_static(int precision, int Nr_d, int Nphi, const void* rho2d, const void* dF_deps_zsum, void* dF_drho,
                           double eps0, double eps_h, double filt_sigma, double beta, double eta, void* stream);

/* Failure detector: ZDA_E_NAN if any E component holds a non-finite value.  Synchronises. */
ZDA_API int zda_check_finite(zda_zone* z);

/* Accounting for bench.py's roofline: bytes per TIME STEP that the zone's current launch plan moves through HBM in run
 * `which` (ZDA_FWD | ZDA_ADJ) when every halo re-read hits L2.  out: host, 5 doubles = { fields (each read once and written
 * once per pass; a pass is one step, or two with ZDA_KERNEL_FUSED2), CPML psi (slabs only), dt/eps (material planes), DFT
 * accumulators incl. the ring copies of E (visit period as planned), halo re-reads if NONE of them hit L2 (upper bound) }. */
ZDA_API int zda_schedule_bytes(zda_zone* z, int which, double* out);

/* Bookkeeping for bench.py: kernels launched by this zone since creation. */
ZDA_API long long zda_launch_count(const zda_zone* z);

/* Name and launch geometry of the time-loop kernel the zone will use ("split" / "fused"). */
ZDA_API const char* zda_kernel_name(const zda_zone* z);

/* a10: zone scheduler -- a full gradient evaluation (forward, adjoint source, adjoint, gradient)
 * of each zone in turn on their streams, zones back to back on the one GPU.
 * Objective per zone: the focal intensity where zda_set_focal_weights was called, else the monitor energy.
 * The zones are driven phase by phase (all forward runs, then each adjoint source followed by its adjoint run, then
 * the gradients), so zones created on DIFFERENT streams overlap on the GPU: that is how zones smaller than one wave of
 * CTAs (the paper's thin wedges) fill the machine; zones on one stream run back to back.  The zones must
 * have pairwise separate workspaces (ZDA_E_BADARG otherwise: a resident zone's tables, materials and sheets live in its
 * workspace; to reuse one buffer down a list, create, solve and destroy the zones one at a time).
 * F_out: host, n_zones doubles (or NULL).  dF_drho[z] / dF_deps_zsum[z]: per-zone device outputs
 * (arrays of n_zones pointers, entries or the arrays themselves may be NULL). */
ZDA_API int zda_lens_gradient(zda_zone** zones, int n_zones, const int* n_steps_fwd, const int* n_steps_adj,
                      const double* adj_t0, const double* adj_sigma_t,
                      double* F_out, void** dF_deps_zsum, void** dF_drho);

/* The lens objective of the paper (PAPER.md:25, 33: the zones' fields add up; :76 "a normally incident plane wave can
 * be decomposed into m = +-1 components"; Eq. 7-8 :78-81; R20, R23): every zone -- and the m = +1 and m = -1
 * members of a pair, which are two zones here -- contributes S_f to ONE focal field, F = sum_f u_f |sum_zones S_f|^2.
 * Forward runs of all zones, the sum, then per zone the adjoint source with u_f conj(S_total_f) g / W, the adjoint run
 * and the gradient; zones on different streams overlap.  All zones need zda_set_focal_weights, the same n_freq and
 * pairwise separate workspaces (else ZDA_E_STATE / ZDA_E_BADARG).  u: host, n_freq doubles (NULL = ones; replaces the
 * per-zone u).  F_out: host, 1 double; S_out: host, 2 n_freq doubles (re, im) -- either may be NULL.  Gradient outputs as
 * in zda_lens_gradient; the gradient of a structure shared by the members of a pair is the sum of theirs. */
ZDA_API int zda_lens_focal_gradient(zda_zone** zones, int n_zones, const int* n_steps_fwd, const int* n_steps_adj,
                            const double* adj_t0, const double* adj_sigma_t, const double* u, double* F_out,
                            double* S_out, void** dF_deps_zsum, void** dF_drho);

#ifdef __cplusplus
}
#endif
#endif /* ZDA_H_ */
