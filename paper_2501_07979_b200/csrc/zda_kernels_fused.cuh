// Fused time-loop kernel: ONE pass per time step.  Each CTA owns a (TI x TJ) tile of (r, phi) and marches
// along z over a chunk of planes; per plane it computes H^{n+1/2}(k) from E^n(k), E^n(k+1) and then
// E^{n+1}(k) from H^{n+1/2}(k), H^{n+1/2}(k-1), so every field is read once and written once per step
// (a3 + a4 of SURVEY 8a in one sweep; CPML, phi phase, source sheet and running DFT fused in).
//
//   * loads: TMA (cp.async.bulk.tensor.4d) halo tiles of E and H into shared-memory rings, signalled on
//     mbarriers, two planes ahead of the compute; r and z out-of-bounds elements are zero-filled by the
//     TMA unit, which IS the PEC ghost (R7); phi ghosts come from the ghost rows of the field layout.
//   * each thread owns 16 bytes along r (4 float / 2 complex-float or double / 1 complex-double), so all
//     shared-memory and global accesses are 128-bit and coalesced.
//   * H on the low halo (row j0-1 and column i0-1) is recomputed by the CTA that needs it, from the OLD
//     buffers (fields and H-side psi are double-buffered), with the same expressions as its owner.
//   * warp w = 1..TJ owns tile row w; warp 0 recomputes the halo row (Hr, Hz) and the halo column (Hphi, Hz).
//
// The per-voxel arithmetic is h_update_voxel / e_update_voxel of zda_device.cuh, shared with the split
// kernels, so the fp64 build (-fmad=false) evaluates exactly the expressions DESIGN.md fixes.
#pragma once
#include <cuda.h>
#include <algorithm>
#include <string>
#include "zda_common.h"
#include "zda_device.cuh"

namespace zda {

constexpr int FUSED_TJ = 7;            // tile rows per CTA (one warp each) + 1 halo warp = 8 warps: two CTAs per SM put
                                       // 4 warps on each SM sub-partition, i.e. 128 registers per thread
constexpr int FUSED_TJ_MIN = 6;        // instantiated tile heights: 6 and 7 (FusedPlan::choose_tj)
constexpr int FUSED_ROW_BYTES = 544;   // 34 x 16 B: [halo unit | 32 payload units | halo unit]
constexpr int FUSED_PAY_BYTES = 512;

template <class T> struct alignas(16) VecT {
    static constexpr int N = 16 / (int)sizeof(T);
    T v[N];
};

template <int TJ> struct alignas(1024) FusedSmem {
    struct alignas(128) Slot { unsigned char c[3][TJ + 2][FUSED_ROW_BYTES]; };
    Slot E[3];                                              // ring over planes k, k+1, k+2
    Slot H[2];                                              // ring over planes k, k+1 (old H)
    alignas(16) unsigned char Hn[2][2][TJ + 1][FUSED_PAY_BYTES];   // new {Hr, Hz} rows, double-buffered over k
    alignas(16) unsigned char Hcol[2][2][TJ][16];                  // new {Hphi, Hz} on the halo column i0 - 1
    alignas(16) unsigned char coef[12][FUSED_PAY_BYTES];           // per-r tables of the tile (Real[TI]): 6 curl coefficients, 6 r-CPML
                                                                   // (an exact-PML zone, R25, appends 6 more BEHIND this struct)
    unsigned long long barE[3], barH[2];
};

struct FusedGeom {
    int n_ti, n_tj, n_zc, chunk;   // tiles in r, phi; z-chunks and their length
    int aE, aH;                    // tensor-map array index of the INPUT E[.][0], H[.][0]
    int cluster, n_tjc;            // thread-block cluster: `cluster` phi-neighbouring tiles marching in lock step (their
                                   // halo rows then meet in L2); n_tjc = ceil(n_tj / cluster)
};

// ---- PTX helpers -------------------------------------------------------------------------------
__device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned long long* bar, unsigned count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(unsigned long long* bar, unsigned bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long* bar, unsigned parity) {
    const unsigned a = smem_u32(bar);
    unsigned ok = 0;
    while (!ok) {
        asm volatile(
            "{\n\t.reg .pred p;\n\t"
            "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
            "selp.u32 %0, 1, 0, p;\n\t}"
            : "=r"(ok) : "r"(a), "r"(parity) : "memory");
    }
}
__device__ __forceinline__ void tma_load_4d(void* dst, const CUtensorMap* map, unsigned long long* bar,
                                            int c0, int c1, int c2, int c3) {
    asm volatile(
        "cp.async.bulk.tensor.4d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4, %5}], [%6];"
        ::"r"(smem_u32(dst)), "l"(map), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(smem_u32(bar)) : "memory");
}

template <class T> __device__ __forceinline__ VecT<T> lds_vec(const unsigned char* row, int unit) {
    return *reinterpret_cast<const VecT<T>*>(row + 16 * unit);
}
template <class T> __device__ __forceinline__ T lds_elem(const unsigned char* row, int unit, int e) {
    return reinterpret_cast<const T*>(row + 16 * unit)[e];
}
template <class T> __device__ __forceinline__ VecT<T> ldg_vec(const T* p) { return *reinterpret_cast<const VecT<T>*>(p); }
template <class T> __device__ __forceinline__ void stg_vec(T* p, const VecT<T>& v) { *reinterpret_cast<VecT<T>*>(p) = v; }

// store the 16-byte group starting at column i < Nr.  A group that straddles Nr also writes the row padding
// [Nr, pitch), which no kernel reads (the tensor map ends at Nr) and which only ever receives finite values.
template <class T> __device__ __forceinline__ void store_row(T* rowp, int i, int, const VecT<T>& v) { stg_vec(rowp + i, v); }

// Loads that must be ISSUED where they are written (before an mbarrier wait), not sunk to their first use:
// volatile asm keeps its order relative to the other volatile asm statements (the mbarrier polls).
template <class X> __device__ __forceinline__ X ldg_early(const X* p) {
    static_assert(sizeof(X) == 4 || sizeof(X) == 8 || sizeof(X) == 16 || sizeof(X) == 32, "unsupported early-load size");
    X out;
    unsigned* w = reinterpret_cast<unsigned*>(&out);
    if constexpr (sizeof(X) == 4) {
        asm volatile("ld.global.u32 %0, [%1];" : "=r"(w[0]) : "l"(p));
    } else if constexpr (sizeof(X) == 8) {
        asm volatile("ld.global.v2.u32 {%0, %1}, [%2];" : "=r"(w[0]), "=r"(w[1]) : "l"(p));
    } else if constexpr (sizeof(X) == 16) {
        asm volatile("ld.global.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(w[0]), "=r"(w[1]), "=r"(w[2]), "=r"(w[3]) : "l"(p));
    } else {
        asm volatile("ld.global.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(w[0]), "=r"(w[1]), "=r"(w[2]), "=r"(w[3]) : "l"(p));
        asm volatile("ld.global.v4.u32 {%0, %1, %2, %3}, [%4];"
                     : "=r"(w[4]), "=r"(w[5]), "=r"(w[6]), "=r"(w[7]) : "l"(reinterpret_cast<const char*>(p) + 16));
    }
    return out;
}

// split-phase cluster barrier: keeps the CTAs of a cluster within one plane of each other without stalling on it
__device__ __forceinline__ void cluster_arrive() { asm volatile("barrier.cluster.arrive.relaxed.aligned;" ::: "memory"); }
__device__ __forceinline__ void cluster_wait() { asm volatile("barrier.cluster.wait.aligned;" ::: "memory"); }

__device__ __forceinline__ void prefetch_l2(const void* p) { asm volatile("prefetch.global.L2 [%0];" ::"l"(p)); }

// VEC consecutive DFT accumulators (complex) of one component: 16 or 32 bytes, 16-byte aligned
template <class R, int VEC> struct alignas(16) DftV { Cx<R> v[VEC]; };
// d[c * stride + e] = (d[c * stride + e] + twp * o_c[e]) + tw * n_c[e], c = 0..2 (o = E of the previous step or
// zero, n = E of this step): all loads first, then the adds in step order, then the stores
template <class T, class R, int VEC>
__device__ __forceinline__ void dft_accumulate(Cx<R>* d, size_t stride, Cx<R> twp, const VecT<T>& o0, const VecT<T>& o1,
                                               const VecT<T>& o2, Cx<R> tw, const VecT<T>& n0, const VecT<T>& n1,
                                               const VecT<T>& n2) {
    using DV = DftV<R, VEC>;
    DV d0 = *reinterpret_cast<const DV*>(d), d1 = *reinterpret_cast<const DV*>(d + stride),
       d2 = *reinterpret_cast<const DV*>(d + 2 * stride);
#pragma unroll
    for (int e = 0; e < VEC; ++e) {
        d0.v[e] = (d0.v[e] + tw_mul(twp, o0.v[e])) + tw_mul(tw, n0.v[e]);
        d1.v[e] = (d1.v[e] + tw_mul(twp, o1.v[e])) + tw_mul(tw, n1.v[e]);
        d2.v[e] = (d2.v[e] + tw_mul(twp, o2.v[e])) + tw_mul(tw, n2.v[e]);
    }
    *reinterpret_cast<DV*>(d) = d0;
    *reinterpret_cast<DV*>(d + stride) = d1;
    *reinterpret_cast<DV*>(d + 2 * stride) = d2;
}

__device__ __forceinline__ float shfl_up1(float x) { return __shfl_up_sync(0xffffffffu, x, 1); }
__device__ __forceinline__ double shfl_up1(double x) { return __shfl_up_sync(0xffffffffu, x, 1); }
template <class R> __device__ __forceinline__ Cx<R> shfl_up1(Cx<R> x) { return {shfl_up1(x.x), shfl_up1(x.y)}; }

// CPML slab index along an axis of N cells: 0..lo-1 in the low slab, lo.. in the high slab, -1 outside
__device__ __forceinline__ int slab_index(int q, int N, int lo, int hi) {
    if (q < lo) return q;
    if (q >= N - hi) return lo + (q - (N - hi));
    return -1;
}

}  // namespace zda

#include "zda_kernels_fused_body.cuh"
