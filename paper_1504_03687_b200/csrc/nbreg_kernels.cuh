// nbreg_kernels.cuh -- sm_100a device code of libnbreg (see include/nbreg.h for the contract).
//
//   relayout_kernel   a1  AoS [N][3] FP64 -> internal SoA FP64                    (HBM-bound)
//   predict_kernel    a2  Hermite predictor, FP64 -> predicted record (40 B/body) (HBM-bound)
//   force_kernel      a3-a6  i-block x j-tile pairwise sum + neighbour lists      (FP32 issue-bound)
//   finalize_kernel   a6-a7  fixed-order sum over j-splits, write-back, counters  (tiny)
//
// Predicted record: 40 B per body = ten FP32 values (xh,yh,zh, xl,yl,zl, vx,vy,vz, m), stored
// COMPONENT-MAJOR INSIDE EACH j-TILE: rec[tile][component][TJ].  A tile (256 bodies, 10 KB) is ONE
// contiguous TMA bulk copy, and one warp-uniform LDS.128 hands the force kernel the same component of
// four consecutive j.  Each thread owns PAIRS of i-particles: every FP32 operation of the pair
// arithmetic is one packed FADD2/FMUL2/FFMA2 (sm_100 f32x2) whose j-side operand is a 32-bit scalar
// broadcast to both halves (SASS operand form `R.F32`), so a j value costs one register read and the
// records need no duplication.  x = hi + lo with hi = fl32(x), lo = fl32(x - hi): positions carry 48
// significant bits, so (hi_j - hi_i) + (lo_j - lo_i) is the FP64 difference rounded once to FP32 --
// the pair arithmetic after that is plain FP32.  A warp whose i-particles sit
// close together (relative to their neighbour radii) differences in its OWN frame instead: one add per
// component (see force_kernel).  Small blocks read the FP64 state directly and predict in the kernel.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace nbreg {

constexpr int TJ = 256;        // j-particles per shared-memory tile
constexpr int RECF = 10;       // floats per predicted record (40 B)
#ifndef NBREG_NSTAGE
#define NBREG_NSTAGE 4
#endif
#ifndef NBREG_GROUP_UNROLL
#define NBREG_GROUP_UNROLL 2
#endif
constexpr int NSTAGE = NBREG_NSTAGE;   // tiles in flight per CTA (bulk-copy ring)
constexpr int GROUP_UNROLL = NBREG_GROUP_UNROLL;   // j-groups per iteration of the inner loop
constexpr int TILE_FLOATS = TJ * RECF;
enum { C_XH = 0, C_YH, C_ZH, C_XL, C_YL, C_ZL, C_VX, C_VY, C_VZ, C_M };   // component rows of a tile
constexpr int UNROLL_J = 4;    // j's per neighbour-detection group
constexpr float GHOST_POS = 1.0e15f;   // padding j's sit here with m = 0
constexpr float TINY_H2 = 1.17549435e-38f;  // FLT_MIN: masks exactly the r2 == 0 self pair when h2 <= 0

// ------------------------------------------------------------------ PTX helpers (mbarrier + bulk copy)
__device__ __forceinline__ uint32_t smem_u32(const void *p) {
    return static_cast<uint32_t>(__cvta_generic_to_shared(p));
}
__device__ __forceinline__ void mbar_init(uint64_t *bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void fence_mbar_init() {
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint64_t *bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes)
                 : "memory");
}
// 1-D TMA bulk copy global -> shared, completion counted in bytes on an mbarrier (SASS: UBLKCP).
__device__ __forceinline__ void bulk_g2s(void *dst, const void *src, uint32_t bytes, uint64_t *bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                     smem_u32(dst)),
                 "l"(__cvta_generic_to_global(src)), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity) {
    uint32_t ok;
    do {
        asm volatile(
            "{\n\t.reg .pred p;\n\t"
            "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
            "selp.u32 %0, 1, 0, p;\n\t}"
            : "=r"(ok)
            : "r"(smem_u32(bar)), "r"(parity)
            : "memory");
    } while (!ok);
}
__device__ __forceinline__ void fence_proxy_async_smem() {   // generic-proxy accesses before, async-proxy (TMA) after
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
}
// Kernels of the block chains are launched with programmatic stream serialization (launch_chain in nbreg.cu): the
// grid is placed while its predecessor in the stream drains; nothing the predecessors wrote may be read before
// this wait.  A no-op in an ordinary launch.
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ float rsqrt_sfu(float x) {   // one MUFU.RSQ, no denormal fix-up code
    float y;
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

// Debug builds (-DNBREG_TIMELINE): thread 0 of every CTA stamps %globaltimer at a few points.
#ifdef NBREG_TIMELINE
__device__ unsigned long long *g_timeline = nullptr;      // [CTA][8]
__device__ __forceinline__ void tl_stamp(int cta, int q) {
    if (threadIdx.x == 0 && g_timeline) {
        unsigned long long t;
        asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
        g_timeline[(size_t)cta * 8 + q] = t;
    }
}
#define TL_STAMP(cta, q) tl_stamp(cta, q)
#else
#define TL_STAMP(cta, q)
#endif

// ------------------------------------------------------------------ a1: re-layout
// in: m[N], x0[N][3], v0[N][3], a0[N][3], j0[N][3], t0[N]  ->  soa[14][Ns] (component-major, streamed
// by the predictor) and aos[N][16] (one 128 B line per body: m, x0, v0, a0, j0, t0, 2 pad -- gathered
// by the neighbour-force kernel, which predicts only the listed bodies).
constexpr int AOS_D = 16;
__device__ __forceinline__ void store_body(int64_t j, int64_t Ns, double m, const double *x, const double *v,
                                           const double *a, const double *jk, double t0, double *__restrict__ soa,
                                           double *__restrict__ aos) {
    soa[0 * Ns + j] = m;
    soa[13 * Ns + j] = t0;
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        soa[(1 + c) * Ns + j] = x[c];
        soa[(4 + c) * Ns + j] = v[c];
        soa[(7 + c) * Ns + j] = a[c];
        soa[(10 + c) * Ns + j] = jk[c];
    }
    if (!aos) return;       // the gather copy exists only once a NEXT-2 / NEXT-3 call has asked for it
    double2 *o = reinterpret_cast<double2 *>(aos + j * AOS_D);
    o[0] = make_double2(m, x[0]);     o[1] = make_double2(x[1], x[2]);
    o[2] = make_double2(v[0], v[1]);  o[3] = make_double2(v[2], a[0]);
    o[4] = make_double2(a[1], a[2]);  o[5] = make_double2(jk[0], jk[1]);
    o[6] = make_double2(jk[2], t0);   o[7] = make_double2(0.0, 0.0);
}

// Bodies [jbeg, jend): the pipelined HOST step (nb_step_host) re-lays chunks out as they arrive.
__global__ void __launch_bounds__(256) relayout_kernel(int64_t jbeg, int64_t jend, int64_t Ns,
                                                       const double *__restrict__ m,
                                                       const double *__restrict__ x0, const double *__restrict__ v0,
                                                       const double *__restrict__ a0, const double *__restrict__ j0,
                                                       const double *__restrict__ t0, double *__restrict__ soa,
                                                       double *__restrict__ aos) {
    int64_t j = jbeg + (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= jend) return;
    double x[3], v[3], a[3], jk[3];
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        x[c] = x0[3 * j + c]; v[c] = v0[3 * j + c]; a[c] = a0[3 * j + c]; jk[c] = j0[3 * j + c];
    }
    store_body(j, Ns, m[j], x, v, a, jk, t0[j], soa, aos);
}

// Incremental ingest (NEXT-3; "Send.R" after a block step only the n integrated particles
// changed): the same stores for the bodies idx[0..n).
__global__ void __launch_bounds__(256) update_j_kernel(int32_t n, int64_t Ns, const int32_t *__restrict__ idx,
                                                       const double *__restrict__ m, const double *__restrict__ x0,
                                                       const double *__restrict__ v0, const double *__restrict__ a0,
                                                       const double *__restrict__ j0, const double *__restrict__ t0,
                                                       double *__restrict__ soa, double *__restrict__ aos) {
    const int q = blockIdx.x * blockDim.x + threadIdx.x;
    if (q >= n) return;
    double x[3], v[3], a[3], jk[3];
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        x[c] = x0[3 * q + c]; v[c] = v0[3 * q + c]; a[c] = a0[3 * q + c]; jk[c] = j0[3 * q + c];
    }
    store_body(idx[q], Ns, m[q], x, v, a, jk, t0[q], soa, aos);
}

// Padding bodies N .. Npad-1 of the FP64 state: massless ghosts far away (written once at nb_open; the
// fused force kernel predicts whole tiles, the predictor writes the same ghost into the records).
__global__ void __launch_bounds__(256) ghost_pad_kernel(int64_t N, int64_t Npad, int64_t Ns, double *__restrict__ soa) {
    const int64_t j = N + (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= Npad) return;
#pragma unroll
    for (int c = 0; c < 14; ++c) soa[c * Ns + j] = (c >= 1 && c <= 3) ? (double)GHOST_POS : 0.0;
}

// Build the gather copy from the SoA state (first NEXT-2 / NEXT-3 call on a context).
__global__ void __launch_bounds__(256) soa_to_aos_kernel(int64_t N, int64_t Ns, const double *__restrict__ soa,
                                                         double *__restrict__ aos) {
    const int64_t j = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= N) return;
    double v[14];
#pragma unroll
    for (int c = 0; c < 14; ++c) v[c] = soa[c * Ns + j];
    double2 *o = reinterpret_cast<double2 *>(aos + j * AOS_D);
    o[0] = make_double2(v[0], v[1]);  o[1] = make_double2(v[2], v[3]);
    o[2] = make_double2(v[4], v[5]);  o[3] = make_double2(v[6], v[7]);
    o[4] = make_double2(v[8], v[9]);  o[5] = make_double2(v[10], v[11]);
    o[6] = make_double2(v[12], v[13]); o[7] = make_double2(0.0, 0.0);
}

// ------------------------------------------------------------------ a2: predictor
// xp = x0 + v0 dt + a0 dt^2/2 + j0 dt^3/6,  vp = v0 + a0 dt + j0 dt^2/2   (reading R2)
__device__ __forceinline__ float *rec_slot(float *rec, int64_t j) {      // &rec[tile][0][j % TJ]
    return rec + (j / TJ) * TILE_FLOATS + (j % TJ);
}
__device__ __forceinline__ const float *rec_slot(const float *rec, int64_t j) {
    return rec + (j / TJ) * TILE_FLOATS + (j % TJ);
}

// One component of the Taylor predictor, FP64.  The jerk term is rounded on its own (not fused) so
// that for dyadic inputs with j0 = 6 q the product rounds back to q dt^3 exactly and the whole sum is
// exact (tests: bitwise vs oracle).  Used by predict_kernel (all j) and irregular_kernel (listed j).
__device__ __forceinline__ double taylor_c2(double dt) { return 0.5 * (dt * dt); }                  // dt^2/2: exact for dyadic dt
__device__ __forceinline__ double taylor_c3(double dt) { return (dt * dt * dt) * (1.0 / 6.0); }     // dt^3/6: the only inexact coefficient
__device__ __forceinline__ void predict_component(double x, double v, double a, double jk, double dt, double c2,
                                                  double c3, double &xp, double &vp) {
    const double p3 = __dmul_rn(jk, c3);
    xp = __dadd_rn(fma(a, c2, fma(v, dt, x)), p3);
    vp = fma(jk, c2, fma(a, dt, v));
}

// Bodies [jbeg, jend) with jend <= Npad; j >= N are the ghost padding.
__global__ void __launch_bounds__(256) predict_kernel(int64_t jbeg, int64_t jend, int64_t N, int64_t Ns, double t,
                                                      const double *__restrict__ soa, float *__restrict__ rec) {
    int64_t j = jbeg + (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= jend) return;
    float *r = rec_slot(rec, j);
    if (j >= N) {   // ghost padding: massless, far away, never a neighbour, contributes exactly 0
        r[C_XH * TJ] = r[C_YH * TJ] = r[C_ZH * TJ] = GHOST_POS;
        r[C_XL * TJ] = r[C_YL * TJ] = r[C_ZL * TJ] = 0.f;
        r[C_VX * TJ] = r[C_VY * TJ] = r[C_VZ * TJ] = 0.f;
        r[C_M * TJ] = 0.f;
        return;
    }
    const double dt = t - soa[13 * Ns + j];
    const double c2 = taylor_c2(dt), c3 = taylor_c3(dt);
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        double xp, vp;
        predict_component(soa[(1 + c) * Ns + j], soa[(4 + c) * Ns + j], soa[(7 + c) * Ns + j],
                          soa[(10 + c) * Ns + j], dt, c2, c3, xp, vp);
        const float hi = __double2float_rn(xp);
        r[(C_XH + c) * TJ] = hi;
        r[(C_XL + c) * TJ] = __double2float_rn(xp - (double)hi);
        r[(C_VX + c) * TJ] = __double2float_rn(vp);
    }
    r[C_M * TJ] = __double2float_rn(soa[j]);
}

__global__ void __launch_bounds__(256) unpack_predicted_kernel(int64_t N, const float *__restrict__ rec,
                                                               double *__restrict__ xp, double *__restrict__ vp) {
    int64_t j = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= N) return;
    const float *r = rec_slot(rec, j);
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        xp[3 * j + c] = (double)r[(C_XH + c) * TJ] + (double)r[(C_XL + c) * TJ];
        vp[3 * j + c] = (double)r[(C_VX + c) * TJ];
    }
}

// a3 for the pipelined HOST step: the active particles' own predicted records, from their FP64
// state, into irec[RECF][n_i_pad].  Same arithmetic
// as predict_kernel, so irec[.][k] is bitwise the record of body idx_i[k] (reading R3: r = 0 exactly
// for the self pair) -- without waiting for the chunk that holds body idx_i[k] to arrive.
// AOS = false: ist is the gathered copy [14][n_i]; AOS = true: the six pointers are the caller's own
// arrays (m[N], x0[N][3], ..., t0[N]; pinned host memory read through the bus, or device memory) and
// the kernel gathers rows idx_i[k] itself.
struct IStateSrc {
    const double *ist;                                       // AOS = false
    const double *m, *x0, *v0, *a0, *j0, *t0;                // AOS = true
    const int32_t *idx_i;
};
template <bool AOS>
__global__ void __launch_bounds__(256) predict_i_kernel(int32_t n_i, int32_t n_i_pad, double t, const IStateSrc src,
                                                        float *__restrict__ irec) {
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= n_i) return;
    double m, t0, x[3], v[3], a[3], jk[3];
    if (AOS) {
        const int64_t i = src.idx_i[k];
        m = src.m[i]; t0 = src.t0[i];
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            x[c] = src.x0[3 * i + c]; v[c] = src.v0[3 * i + c]; a[c] = src.a0[3 * i + c]; jk[c] = src.j0[3 * i + c];
        }
    } else {
        const double *ist = src.ist;
        m = ist[k]; t0 = ist[(size_t)13 * n_i + k];
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            x[c] = ist[(size_t)(1 + c) * n_i + k]; v[c] = ist[(size_t)(4 + c) * n_i + k];
            a[c] = ist[(size_t)(7 + c) * n_i + k]; jk[c] = ist[(size_t)(10 + c) * n_i + k];
        }
    }
    const double dt = t - t0;
    const double c2 = taylor_c2(dt), c3 = taylor_c3(dt);
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        double xp, vp;
        predict_component(x[c], v[c], a[c], jk[c], dt, c2, c3, xp, vp);
        const float hi = __double2float_rn(xp);
        irec[(size_t)(C_XH + c) * n_i_pad + k] = hi;
        irec[(size_t)(C_XL + c) * n_i_pad + k] = __double2float_rn(xp - (double)hi);
        irec[(size_t)(C_VX + c) * n_i_pad + k] = __double2float_rn(vp);
    }
    irec[(size_t)C_M * n_i_pad + k] = __double2float_rn(m);
}

// ------------------------------------------------------------------ a3: spatial order of a large active block
// The local frame of force_kernel needs the 64 i-particles of a warp to sit close together.  A block
// arrives in the caller's order (NBODY6++GPU: the step-sorted list, P:89 -- not spatial), so for large
// blocks the library sorts the SLOTS of the block along a Morton curve of the predicted positions:
// bounding box (integer atomics on ordered keys: order-independent), 42-bit keys (14 bits per axis on
// the box), ties broken by k, bitonic sort (no atomics: the permutation is a pure function of the
// inputs, so results stay bitwise reproducible).
__device__ __forceinline__ uint32_t ordered_u32(float x) {             // monotone map float -> uint32
    const uint32_t b = __float_as_uint(x);
    return (b >> 31) ? ~b : (b | 0x80000000u);
}
__device__ __forceinline__ float ordered_to_float(uint32_t k) {
    return __uint_as_float((k >> 31) ? (k & 0x7fffffffu) : ~k);
}
__device__ __forceinline__ unsigned long long spread21(uint32_t v) {   // bit i -> bit 3 i
    unsigned long long x = v & 0x1fffffu;
    x = (x | x << 32) & 0x1f00000000ffffull;
    x = (x | x << 16) & 0x1f0000ff0000ffull;
    x = (x | x << 8) & 0x100f00f00f00f00full;
    x = (x | x << 4) & 0x10c30c30c30c30c3ull;
    x = (x | x << 2) & 0x1249249249249249ull;
    return x;
}
__device__ __forceinline__ const float *irec_or_rec(const float *rec, const float *irec, const int32_t *idx_i, int k,
                                                    int64_t n_i_pad, int64_t &cs) {
    cs = irec ? n_i_pad : TJ;
    return irec ? irec + k : rec_slot(rec, idx_i ? idx_i[k] : k);
}

// box[0..2] = min of ordered(x), box[3..5] = min of ~ordered(x) (i.e. the maximum), all initialised to ~0.
__global__ void __launch_bounds__(256) block_bbox_kernel(int32_t n_i, int64_t n_i_pad, const int32_t *__restrict__ idx_i,
                                                         const float *__restrict__ rec, const float *__restrict__ irec,
                                                         uint32_t *__restrict__ box) {
    uint32_t lo[3] = {~0u, ~0u, ~0u}, hi[3] = {~0u, ~0u, ~0u};
    for (int k = blockIdx.x * blockDim.x + threadIdx.x; k < n_i; k += gridDim.x * blockDim.x) {
        int64_t cs;
        const float *r = irec_or_rec(rec, irec, idx_i, k, n_i_pad, cs);
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            const uint32_t o = ordered_u32(r[(C_XH + c) * cs]);
            lo[c] = min(lo[c], o); hi[c] = min(hi[c], ~o);
        }
    }
#pragma unroll
    for (int c = 0; c < 3; ++c) {
#pragma unroll
        for (int off = 16; off > 0; off >>= 1) {
            lo[c] = min(lo[c], __shfl_xor_sync(0xffffffffu, lo[c], off));
            hi[c] = min(hi[c], __shfl_xor_sync(0xffffffffu, hi[c], off));
        }
        if ((threadIdx.x & 31) == 0) { atomicMin(box + c, lo[c]); atomicMin(box + 3 + c, hi[c]); }
    }
}

// keys[s] for the n2 = 2^m >= n_i slots of the sort: (42-bit Morton code of the position on the block's
// bounding box, 14 bits per axis) << 22 | k -- ONE 64-bit compare orders by cell and breaks ties by k, and
// after the sort perm[slot] = key & PERM_MASK.  Slots >= n_i sort to the end.  (k < 2^22: blocks of up to
// 4M particles; larger blocks are not reordered.)
constexpr int PERM_BITS = 22;
constexpr unsigned long long PERM_MASK = (1ull << PERM_BITS) - 1;
__device__ __forceinline__ int32_t perm_slot(const unsigned long long *perm, int slot) {
    return (int32_t)(perm[slot] & PERM_MASK);
}
__global__ void __launch_bounds__(256) morton_key_kernel(int32_t n_i, int32_t n2, int64_t n_i_pad,
                                                         const int32_t *__restrict__ idx_i, const float *__restrict__ rec,
                                                         const float *__restrict__ irec, const uint32_t *__restrict__ box,
                                                         unsigned long long *__restrict__ keys) {
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= n2) return;
    if (k >= n_i) { keys[k] = ~0ull; return; }
    int64_t cs;
    const float *r = irec_or_rec(rec, irec, idx_i, k, n_i_pad, cs);
    unsigned long long key = 0;
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const float mn = ordered_to_float(box[c]), mx = ordered_to_float(~box[3 + c]);
        const float ext = mx - mn;
        const float u = ext > 0.f ? (r[(C_XH + c) * cs] - mn) / ext : 0.f;             // in [0, 1]
        const uint32_t q = min((uint32_t)(u * 16384.0f), 16383u);                       // 14 bits
        key |= spread21(q) << (2 - c);
    }
    keys[k] = (key << PERM_BITS) | (unsigned long long)k;
}

// Bitonic sort of the 64-bit keys, ascending.  SORT_CH keys per CTA live in shared memory (one
// compare-exchange per thread and step); merges across chunks go through global memory.
constexpr int SORT_CH = 2048;
constexpr int SORT_T = 1024;
// MODE 0: full sort of each chunk (sizes 2 .. chunk).  MODE 1: the strides chunk/2 .. 1 of merge size `size`.
template <int MODE>
__global__ void __launch_bounds__(SORT_T) bitonic_chunk_kernel(int32_t n2, int32_t size, unsigned long long *__restrict__ keys) {
    __shared__ unsigned long long sk[SORT_CH];
    const int ch = min(n2, SORT_CH);
    const int base = blockIdx.x * ch;
    for (int e = threadIdx.x; e < ch; e += SORT_T) sk[e] = keys[base + e];
    __syncthreads();
    for (int sz = (MODE == 0 ? 2 : size); sz <= (MODE == 0 ? ch : size); sz <<= 1) {
        for (int stride = min(sz >> 1, ch >> 1); stride > 0; stride >>= 1) {
            for (int e = threadIdx.x; e < (ch >> 1); e += SORT_T) {
                const int lo = 2 * e - (e & (stride - 1)), hi = lo + stride;
                const bool up = ((base + lo) & sz) == 0;
                const unsigned long long ka = sk[lo], kb = sk[hi];
                if ((ka > kb) == up) { sk[lo] = kb; sk[hi] = ka; }
            }
            __syncthreads();
        }
    }
    for (int e = threadIdx.x; e < ch; e += SORT_T) keys[base + e] = sk[e];
}
// One compare-exchange step (merge size `size`, stride >= SORT_CH) in global memory.
__global__ void __launch_bounds__(256) bitonic_global_kernel(int32_t n2, int32_t size, int32_t stride,
                                                            unsigned long long *__restrict__ keys) {
    const int e = blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= (n2 >> 1)) return;
    const int lo = 2 * e - (e & (stride - 1)), hi = lo + stride;
    const bool up = (lo & size) == 0;
    const unsigned long long ka = keys[lo], kb = keys[hi];
    if ((ka > kb) == up) { keys[lo] = kb; keys[hi] = ka; }
}

// ------------------------------------------------------------------ a3-a6: force kernel
// Source of the j-data a CTA streams through its bulk-copy ring:
//   SRC_REC    the predicted records nb_predict_all wrote (40 B/body, one 10 KB bulk copy per tile);
//   SRC_STATE  the FP64 j-state itself (112 B/body, fourteen 2 KB bulk copies per tile): every warp
//              PREDICTS the j's it is about to consume, with the predictor's own arithmetic -- the
//              fused predict + force path of small blocks (one reader per j-tile; no predict launch
//              and no 40 B/body round trip through HBM).
enum { SRC_REC = 0, SRC_STATE = 1 };
constexpr int STATE_D = 14;                                   // doubles per body of the FP64 state
constexpr int STATE_TILE_DOUBLES = STATE_D * TJ;              // 28 KB per tile
#ifndef NBREG_STATE_NST_JP
#define NBREG_STATE_NST_JP 3
#endif
template <int SRC, bool JP = false> struct SrcCfg;
template <bool JP> struct SrcCfg<SRC_REC, JP> {
    static constexpr int NST = NSTAGE;                                         // stages in the ring
    static constexpr uint32_t STAGE_BYTES = TILE_FLOATS * sizeof(float);       // 10 KB
    static constexpr int SLICE_COMP = 3;                                       // x', y', z' per j of the warp's share
};
template <bool JP> struct SrcCfg<SRC_STATE, JP> {
    static constexpr int NST = JP ? NBREG_STATE_NST_JP : 2;    // 28 KB stages: what two CTAs per SM leave room for
    static constexpr uint32_t STAGE_BYTES = STATE_TILE_DOUBLES * sizeof(double);   // 28 KB
    static constexpr int SLICE_COMP = RECF;                                    // a whole record per j of the warp's share
};

struct ForceParams {
    const float *rec;             // SRC_REC: predicted records, [Npad / TJ][RECF][TJ]
    const double *soa;            // SRC_STATE: FP64 state [14][Ns] (padding bodies are massless ghosts)
    int64_t Ns;
    double t;                     // SRC_STATE: time to predict to
    const int32_t *idx_i;         // [n_i], or NULL: the block is 0..n_i-1
    const double *h2_i;           // [n_i]; or [N] indexed by body when h2_by_body; or NULL: every h2 = 0
    int32_t h2_by_body;
    const unsigned long long *perm;   // NULL, or sorted keys of a block the library put in Morton order: slot -> k = key & PERM_MASK
    int32_t n_i;
    int32_t n_i_pad;              // n_i rounded up to the CTA's i-block
    const float *irec;            // NULL, or the active particles' own records [RECF][n_i_pad] (nb_step_host, shards)
    int32_t tile0;                // first j-tile of this launch (0 unless the j-range arrives in chunks)
    int32_t ntiles;               // end of this launch's j-tile range (Npad / TJ for a whole pass)
    int32_t split0;               // first row of `partial` this launch writes
    int32_t j_offset;             // global index of this context's body 0 (j-sharding; 0 otherwise): list entries and
                                  // the self test use global indices, idx_i is global when irec is given
    int32_t tiles_per_split;      // contiguous tiles per blockIdx.y
    int32_t cap;
    float g2;                     // local-frame guard: a warp differences in its own frame iff every one of its
                                  // i has |x_i - c|^2 <= g2 * h2_i (c = centre of the warp's bounding box); 0: never
    int32_t *cnt;                 // [>= n_i] neighbour counters, zero on entry (finalize re-zeroes)
    int32_t *nblist;              // caller's [n_i][cap], or NULL: neighbours are only counted
    double *partial;              // [S][7][n_i_pad]
    unsigned int *stats;          // NULL, or {warps in the local frame, warps} (diagnostics; integer atomics)
    const double *blk_dev;        // NULL, or the block descriptor {t_next, n_active, n_regular, status} written by
                                  // select_block_kernel: a SPECULATIVE launch of nb_block_step / nb_ac_step -- the block's
                                  // time and size come from device memory and the launch is a no-op unless status = 1
};
// Status of a selected block: may the speculative chain enqueued behind the selection integrate it?
enum { BLK_SKIPPED = 0, BLK_SPECULATIVE = 1, BLK_NEEDS_HOST = 2, BLK_PAST_T_STOP = 3 };
// The block a speculative launch works on: false = nothing to do.  n and t are overwritten from blk_dev.
__device__ __forceinline__ bool spec_block(const double *blk_dev, int32_t &n, double &t) {
    if (!blk_dev) return true;
    if (blk_dev[3] != (double)BLK_SPECULATIVE) return false;
    t = blk_dev[0];
    n = (int32_t)blk_dev[1];
    return true;
}

// Two active particles (halves .x / .y) held in registers, NEGATED so that every difference is one
// packed add:  d = j + (-i).  Local frame: nxh.. hold -(x_i - c) and the lo parts are unused.
struct IPair {
    float2 nxh, nyh, nzh, nxl, nyl, nzl, nvx, nvy, nvz, h2;
};

#ifdef NBREG_SCALAR_MATH
__device__ __forceinline__ float2 padd(float2 a, float2 b) { return make_float2(__fadd_rn(a.x, b.x), __fadd_rn(a.y, b.y)); }
__device__ __forceinline__ float2 pmul(float2 a, float2 b) { return make_float2(__fmul_rn(a.x, b.x), __fmul_rn(a.y, b.y)); }
__device__ __forceinline__ float2 pfma(float2 a, float2 b, float2 c) { return make_float2(__fmaf_rn(a.x, b.x, c.x), __fmaf_rn(a.y, b.y, c.y)); }
#else
__device__ __forceinline__ float2 padd(float2 a, float2 b) { return __fadd2_rn(a, b); }
__device__ __forceinline__ float2 pmul(float2 a, float2 b) { return __fmul2_rn(a, b); }
__device__ __forceinline__ float2 pfma(float2 a, float2 b, float2 c) { return __ffma2_rn(a, b, c); }
#endif
__device__ __forceinline__ float2 bc(float s) { return make_float2(s, s); }   // -> scalar `R.F32` operand
__device__ __forceinline__ float pick(const float4 &v, int u) { return u == 0 ? v.x : u == 1 ? v.y : u == 2 ? v.z : v.w; }
// j-side operand number u of a group of four consecutive j.  JP = false: j number u broadcast to both
// halves (the halves are two i).  JP = true (tiny blocks): the halves are the two consecutive j 2u, 2u+1
// against ONE i held in both halves of the i registers -- a warp then covers 32 i instead of 64.
template <bool JP>
__device__ __forceinline__ float2 jop(const float4 &v, int u) {
    if constexpr (JP) return u == 0 ? make_float2(v.x, v.y) : make_float2(v.z, v.w);
    else return bc(pick(v, u));
}

// One neighbour of active particle k: take a slot of its row with an integer atomic (rows are shared
// with the other j-splits and warps); entries past the capacity are only counted (reading R9).
__device__ __forceinline__ void append_one(int32_t k, int32_t jg, int32_t cap, int32_t *cnt, int32_t *nblist) {
    const int32_t pos = atomicAdd(cnt + k, 1);
    if (pos < cap && nblist) nblist[(int64_t)k * cap + pos] = jg;
}

// The seven FP32 partial sums of one i-pair over (a share of) one j-tile.
struct Acc7 {
    float2 ax, ay, az, jx, jy, jz, ph;
};

// Pair terms of one j against an i-pair, after r^2 is known.  MASKED = false is the fast path (no
// lane of the warp has a neighbour or its self pair among the group's j's): plain MUFU.RSQ, no
// predicates.  MASKED = true drops the pairs with r2 < h2 by zeroing 1/r BEFORE any product (no inf*0).
template <bool MASKED>
__device__ __forceinline__ void pair_terms(Acc7 &A, const IPair &I, float2 dx, float2 dy, float2 dz, float2 r2,
                                           float2 rinv, float2 jvx, float2 jvy, float2 jvz, float2 jm) {
    const float2 dvx = padd(jvx, I.nvx);
    const float2 dvy = padd(jvy, I.nvy);
    const float2 dvz = padd(jvz, I.nvz);
    const float2 rv = pfma(dz, dvz, pfma(dy, dvy, pmul(dx, dvx)));
    if (MASKED) {       // a select, not a product: the self pair's rsqrt(0) = inf never reaches the arithmetic
        rinv.x = r2.x < I.h2.x ? 0.f : rinv.x;
        rinv.y = r2.y < I.h2.y ? 0.f : rinv.y;
    }
    const float2 rinv2 = pmul(rinv, rinv);
    const float2 mrinv = pmul(jm, rinv);
    const float2 mrinv3 = pmul(mrinv, rinv2);
    const float2 alpha = pmul(pmul(rv, rinv2), make_float2(-3.0f, -3.0f));
    A.ph = padd(A.ph, mrinv);
    A.ax = pfma(mrinv3, dx, A.ax);
    A.ay = pfma(mrinv3, dy, A.ay);
    A.az = pfma(mrinv3, dz, A.az);
    A.jx = pfma(mrinv3, pfma(alpha, dx, dvx), A.jx);
    A.jy = pfma(mrinv3, pfma(alpha, dy, dvy), A.jy);
    A.jz = pfma(mrinv3, pfma(alpha, dz, dvz), A.jz);
}

// Where a warp finds the components of its share of a tile (shared memory, floats).  Positions: px + c * SX
// (LOCAL: x' = x_j - c of the warp; else the hi parts, with the lo parts at pl + c * SX); velocities
// pv + c * SV; masses pm.
struct JPtrs {
    const float *px, *pl, *pv, *pm;
};

// All pairs of the warp's i-pair(s) with SUBN consecutive j of one tile.  LOCAL: positions are already
// differenced against the warp's origin -- ONE packed add per component (27 packed FP32 instructions
// per 2 i x 1 j); otherwise hi/lo differencing, three adds per component (33).
// j-packed variants, tiny blocks (js = 2, 4: a CTA with at most 16 / 8 active particles): the lanes of the warp
// are js groups of 32 / js; group q holds the same 32 / js i-particles and takes the q-th part of the SUBN
// j's, so the addresses are uniform per group (one LDS.128 wavefront: the groups read different 16 B pieces
// of the same rows) and the padded pair work shrinks from 32 to 16 / 8 i-slots.
template <bool LOCAL, bool JP, int SUBN, int SX, int SV, bool GROUPED = false>
__device__ __forceinline__ void tile_pairs(Acc7 &A, const IPair &I, JPtrs P, int32_t jbase,
                                           const int32_t (&my_idx)[2], const int32_t (&my_k)[2],
                                           const ForceParams &p, int js = 1, int q = 0) {
    constexpr int NU = JP ? 2 : 4;           // packed iterations per group of four j
    static_assert(!GROUPED || (JP && SUBN % (4 * UNROLL_J) == 0), "lane groups along j: j-packed, up to four per warp");
    int span = SUBN;                         // j's of this lane (a compile-time constant unless GROUPED)
    if constexpr (GROUPED) {
        span = SUBN / js;
        const int off = q * span;
        P.px += off; P.pv += off; P.pm += off;
        if constexpr (!LOCAL) P.pl += off;
        jbase += off;
    }
#pragma unroll GROUP_UNROLL
    for (int g = 0; g < span; g += UNROLL_J) {
        // warp-uniform addresses: LDS.128 broadcasts of one component of 4 consecutive j
        float4 cx = *reinterpret_cast<const float4 *>(P.px + g);
        float4 cy = *reinterpret_cast<const float4 *>(P.px + SX + g);
        float4 cz = *reinterpret_cast<const float4 *>(P.px + 2 * SX + g);
        float4 lx, ly, lz;
        if constexpr (!LOCAL) {
            lx = *reinterpret_cast<const float4 *>(P.pl + g);
            ly = *reinterpret_cast<const float4 *>(P.pl + SX + g);
            lz = *reinterpret_cast<const float4 *>(P.pl + 2 * SX + g);
        }
        const float4 cvx = *reinterpret_cast<const float4 *>(P.pv + g);
        const float4 cvy = *reinterpret_cast<const float4 *>(P.pv + SV + g);
        const float4 cvz = *reinterpret_cast<const float4 *>(P.pv + 2 * SV + g);
        const float4 cm = *reinterpret_cast<const float4 *>(P.pm + g);
        // phase 1: differences and r^2 of the group's 4 j against the i-pair
        float2 dx[NU], dy[NU], dz[NU], r2[NU], rinv[NU];
#pragma unroll
        for (int u = 0; u < NU; ++u) {
            if constexpr (LOCAL) {
                dx[u] = padd(jop<JP>(cx, u), I.nxh);
                dy[u] = padd(jop<JP>(cy, u), I.nyh);
                dz[u] = padd(jop<JP>(cz, u), I.nzh);
            } else {
                dx[u] = padd(padd(jop<JP>(cx, u), I.nxh), padd(jop<JP>(lx, u), I.nxl));
                dy[u] = padd(padd(jop<JP>(cy, u), I.nyh), padd(jop<JP>(ly, u), I.nyl));
                dz[u] = padd(padd(jop<JP>(cz, u), I.nzh), padd(jop<JP>(lz, u), I.nzl));
            }
            r2[u] = pfma(dz[u], dz[u], pfma(dy[u], dy[u], pmul(dx[u], dx[u])));
            rinv[u].x = rsqrt_sfu(r2[u].x);        // issued before the vote: SFU latency overlaps the test
            rinv[u].y = rsqrt_sfu(r2[u].y);
        }
        // one test per i for the whole group (FMNMX3): a neighbour, or the self pair (r2 == 0)?
        float mn0, mn1;
        if constexpr (JP) {
            mn0 = fminf(r2[0].x, r2[1].x);
            mn1 = fminf(r2[0].y, r2[1].y);
        } else {
            mn0 = fminf(fminf(fminf(r2[0].x, r2[1].x), r2[2].x), r2[3].x);
            mn1 = fminf(fminf(fminf(r2[0].y, r2[1].y), r2[2].y), r2[3].y);
        }
        const bool hit = (mn0 < I.h2.x) | (mn1 < I.h2.y);
        if (!__any_sync(0xffffffffu, hit)) {    // ~95 % of groups at N_b ~ 150, N = 1M: nothing to mask
#pragma unroll
            for (int u = 0; u < NU; ++u)
                pair_terms<false>(A, I, dx[u], dy[u], dz[u], r2[u], rinv[u], jop<JP>(cvx, u), jop<JP>(cvy, u),
                                  jop<JP>(cvz, u), jop<JP>(cm, u));
        } else {
#pragma unroll
            for (int u = 0; u < NU; ++u)
                pair_terms<true>(A, I, dx[u], dy[u], dz[u], r2[u], rinv[u], jop<JP>(cvx, u), jop<JP>(cvy, u),
                                 jop<JP>(cvz, u), jop<JP>(cm, u));
            if (hit) {      // rare: lanes hold different i, each takes slots of its own rows
#pragma unroll
                for (int u = 0; u < NU; ++u) {
                    // half .x / .y of iteration u: (i, j) = (my i 0, j u) / (my i 1, j u), or, j-packed,
                    // (my i, j 2u) / (my i, j 2u + 1)
                    const int32_t jg0 = jbase + g + (JP ? 2 * u : u), jg1 = JP ? jg0 + 1 : jg0;
                    if (r2[u].x < I.h2.x && jg0 != my_idx[0]) append_one(my_k[0], jg0, p.cap, p.cnt, p.nblist);
                    if (r2[u].y < I.h2.y && jg1 != my_idx[1]) append_one(my_k[1], jg1, p.cap, p.cnt, p.nblist);
                }
            }
        }
    }
}

// Shared-memory plan of one force-kernel CTA (host and device use the same numbers).
template <int WI, int WJ, bool JP, int SRC>
struct ForceSmem {
    static constexpr int NW = WI * WJ, NT = 32 * NW, NH = JP ? 1 : 2, SUB = TJ / WJ;
    static constexpr size_t RING = (size_t)SrcCfg<SRC, JP>::NST * SrcCfg<SRC, JP>::STAGE_BYTES;     // bulk-copy ring
    static constexpr size_t SLICES = (size_t)NW * SrcCfg<SRC, JP>::SLICE_COMP * SUB * sizeof(float);   // one per warp
    static constexpr size_t ACC = (size_t)7 * NH * NT * sizeof(double);                     // FP64 running sums
    static constexpr size_t BARS = (size_t)SrcCfg<SRC, JP>::NST * (sizeof(uint64_t) + sizeof(int));
    static constexpr size_t TOTAL = RING + SLICES + ACC + BARS + 64;
    static_assert(WJ == 1 || (size_t)WJ * 7 * 32 * NH * WI * sizeof(double) <= RING + SLICES,
                  "the WJ reduction reuses the ring and the slices");
};

// The Taylor predictor for one body of an FP64 state tile in shared memory ([14][TJ] doubles).
__device__ __forceinline__ void predict_from_tile(const double *st, int b, double t, double (&xp)[3], double (&vp)[3],
                                                  double &m) {
    m = st[b];
    const double dt = t - st[13 * TJ + b];
    const double c2 = taylor_c2(dt), c3 = taylor_c3(dt);
#pragma unroll
    for (int c = 0; c < 3; ++c)
        predict_component(st[(1 + c) * TJ + b], st[(4 + c) * TJ + b], st[(7 + c) * TJ + b], st[(10 + c) * TJ + b], dt,
                          c2, c3, xp[c], vp[c]);
}

// Each thread owns one PAIR of i-particles; WI warps along i (64 i each), WJ warps along j (each
// takes TJ/WJ j's of every tile).  CTA = 32*WI*WJ threads, i-block = 64*WI.
// JP (blocks of <= 32 active particles, and the ragged tail of small blocks): each thread owns ONE
// i-particle and the packed halves are two consecutive j; i-block = 32*WI.
//
// Local frame.  Every warp takes the centre c of the bounding box of ITS i-particles as origin.  If all of
// them satisfy |x_i - c|^2 <= g2 * h2_i the warp re-expresses its share of every j-tile in that frame
// once per tile (x'_j = fl(fl(xh_j - c) + xl_j), into a warp-private slice of shared memory; from the FP64
// state: x'_j = fl(x_j - c)) and the pair loop needs ONE add per component: 27 packed instructions per
// (2 i x 1 j) instead of 33.  Error of the difference: <= 1.8e-7 |dx| + 2.4e-7 |x_i - c| (half of that from
// the FP64 state), and regular pairs have |dx| >= h_i, so the guard bounds the relative error by
// 1.8e-7 + 2.4e-7 sqrt(g2) -- inside the tolerance budget and translation invariant.
// The i-particle is transformed with the same two operations, so its own record still sits at r = 0
// exactly.  A warp that fails the guard (scattered block, h2 <= 0) keeps the hi/lo differencing.
template <int WI, int WJ, int MINB, bool JP = false, int SRC = SRC_REC>
__global__ void __launch_bounds__(32 * WI *WJ, MINB) force_kernel(const ForceParams p) {
    using SM = ForceSmem<WI, WJ, JP, SRC>;
    using SC = SrcCfg<SRC, JP>;
    constexpr int NW = SM::NW, NT = SM::NT, NH = SM::NH, SUB = SM::SUB, NST = SC::NST;
    constexpr int IB = 32 * NH * WI;
    constexpr int SLICE = SC::SLICE_COMP * SUB;
    static_assert(SUB % UNROLL_J == 0 && UNROLL_J == 4, "a group is one LDS.128 per component");

    extern __shared__ __align__(128) unsigned char smem_raw[];
    unsigned char *ring = smem_raw;                                            // [NST][STAGE_BYTES]
    float *slice = reinterpret_cast<float *>(smem_raw + SM::RING) + (threadIdx.x >> 5) * SLICE;   // this warp's
    // FP64 running sums live in shared memory ([7 NH][threads], touched once per flush): the registers
    // go to the pair arithmetic instead.
    double *acc64 = reinterpret_cast<double *>(smem_raw + SM::RING + SM::SLICES) + threadIdx.x;
    uint64_t *full = reinterpret_cast<uint64_t *>(smem_raw + SM::RING + SM::SLICES + SM::ACC);
    int *done = reinterpret_cast<int *>(full + NST);                           // warps finished with a stage

    const int tid = threadIdx.x;
    const int warp = tid >> 5, lane = tid & 31;
    const int wi = warp % WI, wj = warp / WI;
    int32_t n_i = p.n_i;
    double t_pred = p.t;
    pdl_wait();
    if (!spec_block(p.blk_dev, n_i, t_pred)) return;    // (uniform over the grid, before any barrier)
    // j-packed variants: a CTA with <= 16 / 8 active particles (the tiny blocks of the deep levels; the tail
    // of a small block) groups its lanes 2 / 4 ways along j -- decided here, from the block size, so that a
    // speculative launch (n_i from device memory) takes the right mapping too
    int js = 1;
    if constexpr (JP) {
        const int nv = n_i - (int)blockIdx.x * IB;
        js = nv <= 8 ? 4 : nv <= 16 ? 2 : 1;
    }
    const int il = 32 / js, li = lane & (il - 1), lq = lane / il;      // i-slot of the lane, its group along j

    const int tile_begin = p.tile0 + blockIdx.y * p.tiles_per_split;
    const int tile_end = min(tile_begin + p.tiles_per_split, p.ntiles);
    const int ntile = max(tile_end - tile_begin, 0);
    TL_STAMP(blockIdx.y * gridDim.x + blockIdx.x, 0);

    if (tid == 0) {
#pragma unroll
        for (int s = 0; s < NST; ++s) {
            mbar_init(&full[s], 1);
            done[s] = 0;
        }
        fence_mbar_init();
    }
    __syncthreads();

    auto issue = [&](int tile, int s) {     // one tile into stage s, completion counted in bytes on full[s]
        mbar_arrive_expect_tx(&full[s], SC::STAGE_BYTES);
        if constexpr (SRC == SRC_REC) {
            bulk_g2s(ring + (size_t)s * SC::STAGE_BYTES, p.rec + (size_t)tile * TILE_FLOATS, SC::STAGE_BYTES, &full[s]);
        } else {
            double *dst = reinterpret_cast<double *>(ring + (size_t)s * SC::STAGE_BYTES);
#pragma unroll
            for (int c = 0; c < STATE_D; ++c)      // row c of the state: 256 consecutive doubles
                bulk_g2s(dst + c * TJ, p.soa + (size_t)c * p.Ns + (size_t)tile * TJ, TJ * sizeof(double), &full[s]);
        }
    };
    if (tid == NT - 32) {     // the first copies fly while the i-state is gathered (issued by the last warp: warp 0 gathers)
        for (int s = 0; s < NST && s < ntile; ++s) issue(tile_begin + s, s);
    }

    // ---- a3: gather the i-state (the i-particle IS predicted record idx_i[k]; reading R3), choose the frame
    IPair I;
    int32_t my_idx[2], my_k[2];
    bool local;
    float org[3];
    {
        float ph[2][3], pl[2][3], pv[2][3], ph2[2];
        double pd[2][3];
        bool valid[2];
#pragma unroll
        for (int h = 0; h < NH; ++h) {
            const int slot = blockIdx.x * IB + wi * (32 * NH) + h * 32 + li;
            valid[h] = slot < n_i;
            const int k = (valid[h] && p.perm) ? perm_slot(p.perm, slot) : slot;   // caller's numbering: rows, counters, inputs
            my_k[h] = k;
            my_idx[h] = -1;
#pragma unroll
            for (int c = 0; c < 3; ++c) { ph[h][c] = pl[h][c] = pv[h][c] = 0.f; pd[h][c] = 0.0; }
            ph2[h] = TINY_H2;
            // Only the warps with wj == 0 go to global memory: the other WJ - 1 warps of the CTA hold the
            // same i and get the values through shared memory below (every CTA of the grid asks L2 for
            // the same few lines at the same moment; eight times fewer requests shorten that queue).
            if (valid[h] && (WJ == 1 || wj == 0)) {
                const int32_t idx = p.idx_i ? p.idx_i[k] : k;      // NULL = identity block (full-N pass)
                my_idx[h] = idx;
                // h2_i NULL: no neighbours (total force); h2_by_body: the array is indexed by body, not by k
                ph2[h] = p.h2_i ? fmaxf(__double2float_rn(p.h2_i[p.h2_by_body ? idx : k]), TINY_H2) : TINY_H2;
                if constexpr (SRC == SRC_STATE) {                  // the predictor's own arithmetic on body idx
                    const double *s0 = p.soa + idx;
                    const double dt = t_pred - s0[(size_t)13 * p.Ns];
                    const double c2 = taylor_c2(dt), c3 = taylor_c3(dt);
#pragma unroll
                    for (int c = 0; c < 3; ++c) {
                        double xp, vp;
                        predict_component(s0[(size_t)(1 + c) * p.Ns], s0[(size_t)(4 + c) * p.Ns],
                                          s0[(size_t)(7 + c) * p.Ns], s0[(size_t)(10 + c) * p.Ns], dt, c2, c3, xp, vp);
                        pd[h][c] = xp;
                        ph[h][c] = __double2float_rn(xp);
                        pl[h][c] = __double2float_rn(xp - (double)ph[h][c]);
                        pv[h][c] = __double2float_rn(vp);
                    }
                } else {
                    const float *r = p.irec ? p.irec + k : rec_slot(p.rec, idx);
                    const int64_t cs = p.irec ? p.n_i_pad : TJ;    // component stride
#pragma unroll
                    for (int c = 0; c < 3; ++c) {
                        ph[h][c] = r[(C_XH + c) * cs];
                        pl[h][c] = r[(C_XL + c) * cs];
                        pv[h][c] = r[(C_VX + c) * cs];
                    }
                }
            }
        }
        if constexpr (WJ > 1) {
            constexpr int NF = (SRC == SRC_STATE) ? 17 : 11;       // words per (i-warp, half, lane)
            static_assert((size_t)WI * 2 * NF * 32 * sizeof(float) <= SM::ACC, "the exchange uses the (still unused) FP64 sums");
            float *xch = reinterpret_cast<float *>(smem_raw + SM::RING + SM::SLICES) + (size_t)wi * 2 * NF * 32 + lane;
#pragma unroll
            for (int h = 0; h < NH; ++h) {
                float *x = xch + h * NF * 32;
                if (wj == 0) {
#pragma unroll
                    for (int c = 0; c < 3; ++c) { x[c * 32] = ph[h][c]; x[(3 + c) * 32] = pl[h][c]; x[(6 + c) * 32] = pv[h][c]; }
                    x[9 * 32] = ph2[h];
                    x[10 * 32] = __int_as_float(my_idx[h]);
                    if constexpr (SRC == SRC_STATE) {
#pragma unroll
                        for (int c = 0; c < 3; ++c) {
                            x[(11 + 2 * c) * 32] = __int_as_float(__double2hiint(pd[h][c]));
                            x[(12 + 2 * c) * 32] = __int_as_float(__double2loint(pd[h][c]));
                        }
                    }
                }
            }
            __syncthreads();
#pragma unroll
            for (int h = 0; h < NH; ++h) {
                const float *x = xch + h * NF * 32;
                if (wj != 0) {
#pragma unroll
                    for (int c = 0; c < 3; ++c) { ph[h][c] = x[c * 32]; pl[h][c] = x[(3 + c) * 32]; pv[h][c] = x[(6 + c) * 32]; }
                    ph2[h] = x[9 * 32];
                    my_idx[h] = __float_as_int(x[10 * 32]);
                    if constexpr (SRC == SRC_STATE) {
#pragma unroll
                        for (int c = 0; c < 3; ++c)
                            pd[h][c] = __hiloint2double(__float_as_int(x[(11 + 2 * c) * 32]), __float_as_int(x[(12 + 2 * c) * 32]));
                    }
                }
            }
            __syncthreads();                                       // the region becomes the FP64 sums below
        }
        if constexpr (JP) {       // both halves of the registers hold the same i
            my_k[1] = my_k[0]; my_idx[1] = my_idx[0]; valid[1] = valid[0]; ph2[1] = ph2[0];
#pragma unroll
            for (int c = 0; c < 3; ++c) { ph[1][c] = ph[0][c]; pl[1][c] = pl[0][c]; pv[1][c] = pv[0][c]; pd[1][c] = pd[0][c]; }
        }
        // the warp's origin: centre of the bounding box of its valid i (an FP32 number; any value is correct)
        float mn[3], mx[3];
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            mn[c] = 3.0e38f; mx[c] = -3.0e38f;
#pragma unroll
            for (int h = 0; h < 2; ++h)
                if (valid[h]) { mn[c] = fminf(mn[c], ph[h][c]); mx[c] = fmaxf(mx[c], ph[h][c]); }
#pragma unroll
            for (int off = 16; off > 0; off >>= 1) {
                mn[c] = fminf(mn[c], __shfl_xor_sync(0xffffffffu, mn[c], off));
                mx[c] = fmaxf(mx[c], __shfl_xor_sync(0xffffffffu, mx[c], off));
            }
            org[c] = mn[c] <= mx[c] ? __fmul_rn(0.5f, __fadd_rn(mn[c], mx[c])) : 0.f;
        }
        float ip[2][3];
        bool ok = true;
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            float d2 = 0.f;
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                // EXACTLY the operations the staging applies to a j: the particle's own record lands on itself
                if constexpr (SRC == SRC_STATE) ip[h][c] = __double2float_rn(pd[h][c] - (double)org[c]);
                else ip[h][c] = __fadd_rn(__fadd_rn(ph[h][c], -org[c]), pl[h][c]);
                d2 = fmaf(ip[h][c], ip[h][c], d2);
            }
            ok = ok && (!valid[h] || d2 <= p.g2 * ph2[h]);
        }
        local = (p.g2 > 0.f) && __all_sync(0xffffffffu, ok);
        if (p.stats && lane == 0) {
            atomicAdd(p.stats + 1, 1u);
            if (local) atomicAdd(p.stats, 1u);
        }
        float nx[2][3], nl[2][3];
#pragma unroll
        for (int h = 0; h < 2; ++h)
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                // padding lane: far from everything (also from the ghost j's), result discarded
                nx[h][c] = !valid[h] ? GHOST_POS : local ? -ip[h][c] : -ph[h][c];
                nl[h][c] = (!valid[h] || local) ? 0.f : -pl[h][c];
            }
        I.nxh = make_float2(nx[0][0], nx[1][0]); I.nyh = make_float2(nx[0][1], nx[1][1]);
        I.nzh = make_float2(nx[0][2], nx[1][2]); I.nxl = make_float2(nl[0][0], nl[1][0]);
        I.nyl = make_float2(nl[0][1], nl[1][1]); I.nzl = make_float2(nl[0][2], nl[1][2]);
        I.nvx = make_float2(-pv[0][0], -pv[1][0]); I.nvy = make_float2(-pv[0][1], -pv[1][1]);
        I.nvz = make_float2(-pv[0][2], -pv[1][2]); I.h2 = make_float2(ph2[0], ph2[1]);
    }

#pragma unroll
    for (int c = 0; c < 7 * NH; ++c) acc64[c * NT] = 0.0;      // slot h * 7 + c of this thread

    Acc7 A;                   // FP32 partial sums of at most TJ pair terms (WJ tile shares of SUB j each)
    A.ax = A.ay = A.az = A.jx = A.jy = A.jz = A.ph = make_float2(0.f, 0.f);

    // Stage hand-back without a CTA barrier: the LAST warp to finish with stage s refills it, so
    // warps drift up to NST-1 tiles apart instead of meeting at a __syncthreads every tile.
    auto release = [&](int it, int s) {
        __syncwarp();
        if (lane == 0) {
            __threadfence_block();                       // my reads of stage s are done (release)
            if (atomicAdd(&done[s], 1) == NW - 1) {
                done[s] = 0;
                __threadfence_block();
                if (it + NST < ntile) {
                    fence_proxy_async_smem();            // generic reads -> async-proxy overwrite
                    issue(tile_begin + it + NST, s);
                }
            }
        }
    };

    TL_STAMP(blockIdx.y * gridDim.x + blockIdx.x, 1);
    for (int it = 0; it < ntile; ++it) {
        const int s = it % NST;
        mbar_wait(&full[s], (uint32_t)((it / NST) & 1));
        if (it == 0) TL_STAMP(blockIdx.y * gridDim.x + blockIdx.x, 2);
        const int32_t jbase = p.j_offset + (tile_begin + it) * TJ + wj * SUB;

        if constexpr (SRC == SRC_STATE) {
            // predict the j's this warp is about to consume into its slice; the stage is free right after
            const double *st = reinterpret_cast<const double *>(ring + (size_t)s * SC::STAGE_BYTES);
#pragma unroll
            for (int q = lane; q < SUB; q += 32) {
                double xp[3], vp[3], m;
                predict_from_tile(st, wj * SUB + q, t_pred, xp, vp, m);
#pragma unroll
                for (int c = 0; c < 3; ++c) {
                    if (local) {
                        slice[c * SUB + q] = __double2float_rn(xp[c] - (double)org[c]);
                        slice[(3 + c) * SUB + q] = __double2float_rn(vp[c]);
                    } else {
                        const float hi = __double2float_rn(xp[c]);
                        slice[c * SUB + q] = hi;
                        slice[(3 + c) * SUB + q] = __double2float_rn(xp[c] - (double)hi);
                        slice[(6 + c) * SUB + q] = __double2float_rn(vp[c]);
                    }
                }
                slice[(local ? 6 : 9) * SUB + q] = __double2float_rn(m);
            }
            release(it, s);                              // (starts with __syncwarp: the slice is complete)
            if (local) {
                const JPtrs P = {slice, nullptr, slice + 3 * SUB, slice + 6 * SUB};
                if (JP && js > 1) tile_pairs<true, JP, SUB, SUB, SUB, JP>(A, I, P, jbase, my_idx, my_k, p, js, lq);
                else tile_pairs<true, JP, SUB, SUB, SUB>(A, I, P, jbase, my_idx, my_k, p);
            } else {
                const JPtrs P = {slice, slice + 3 * SUB, slice + 6 * SUB, slice + 9 * SUB};
                if (JP && js > 1) tile_pairs<false, JP, SUB, SUB, SUB, JP>(A, I, P, jbase, my_idx, my_k, p, js, lq);
                else tile_pairs<false, JP, SUB, SUB, SUB>(A, I, P, jbase, my_idx, my_k, p);
            }
            __syncwarp();                                // every lane is out of the slice before it is rewritten
        } else {
            const float *tsub = reinterpret_cast<const float *>(ring + (size_t)s * SC::STAGE_BYTES) + wj * SUB;
            if (local) {
                // x'_j = fl(fl(xh_j - c) + xl_j) for the warp's share of the tile (the i got the same two operations)
                if constexpr (SUB >= 128) {
#pragma unroll
                    for (int q = 4 * lane; q < SUB; q += 128)
#pragma unroll
                        for (int c = 0; c < 3; ++c) {
                            const float4 hi = *reinterpret_cast<const float4 *>(tsub + (C_XH + c) * TJ + q);
                            const float4 lo = *reinterpret_cast<const float4 *>(tsub + (C_XL + c) * TJ + q);
                            const float2 no = make_float2(-org[c], -org[c]);
                            const float2 a = padd(padd(make_float2(hi.x, hi.y), no), make_float2(lo.x, lo.y));
                            const float2 b = padd(padd(make_float2(hi.z, hi.w), no), make_float2(lo.z, lo.w));
                            *reinterpret_cast<float4 *>(slice + c * SUB + q) = make_float4(a.x, a.y, b.x, b.y);
                        }
                } else {
#pragma unroll
                    for (int q = lane; q < SUB; q += 32)
#pragma unroll
                        for (int c = 0; c < 3; ++c)
                            slice[c * SUB + q] =
                                __fadd_rn(__fadd_rn(tsub[(C_XH + c) * TJ + q], -org[c]), tsub[(C_XL + c) * TJ + q]);
                }
                __syncwarp();
                const JPtrs P = {slice, nullptr, tsub + C_VX * TJ, tsub + C_M * TJ};
                if (JP && js > 1) tile_pairs<true, JP, SUB, SUB, TJ, JP>(A, I, P, jbase, my_idx, my_k, p, js, lq);
                else tile_pairs<true, JP, SUB, SUB, TJ>(A, I, P, jbase, my_idx, my_k, p);
            } else {
                const JPtrs P = {tsub, tsub + C_XL * TJ, tsub + C_VX * TJ, tsub + C_M * TJ};
                if (JP && js > 1) tile_pairs<false, JP, SUB, TJ, TJ, JP>(A, I, P, jbase, my_idx, my_k, p, js, lq);
                else tile_pairs<false, JP, SUB, TJ, TJ>(A, I, P, jbase, my_idx, my_k, p);
            }
            release(it, s);                              // (its __syncwarp also frees the slice)
        }

        // flush: FP32 partial sums of <= WJ * SUB = TJ terms go into the FP64 running sums
        if ((it + 1) % WJ == 0 || it + 1 == ntile) {
            const float2 *Av = &A.ax;       // ax, ay, az, jx, jy, jz, ph
#pragma unroll
            for (int c = 0; c < 7; ++c) {
                if constexpr (JP) {     // both halves belong to the same i (even / odd j): one sum, fixed order
                    acc64[c * NT] += (double)Av[c].x + (double)Av[c].y;
                } else {
                    acc64[c * NT] += (double)Av[c].x;
                    acc64[(7 + c) * NT] += (double)Av[c].y;
                }
            }
            A.ax = A.ay = A.az = A.jx = A.jy = A.jz = A.ph = make_float2(0.f, 0.f);
        }
    }

    TL_STAMP(blockIdx.y * gridDim.x + blockIdx.x, 3);
    // ---- a6: fixed-order reduction over the WJ warps that shared these i, then one partial per split
    double out64[NH][7];
#pragma unroll
    for (int h = 0; h < NH; ++h)
#pragma unroll
        for (int c = 0; c < 7; ++c) out64[h][c] = acc64[(h * 7 + c) * NT];
    if constexpr (JP) {         // the js lane groups hold shares of the same i: fixed xor tree, every lane gets the sum
        for (int off = il; off < 32; off <<= 1)
#pragma unroll
            for (int c = 0; c < 7; ++c) out64[0][c] += __shfl_xor_sync(0xffffffffu, out64[0][c], off);
    }
    if constexpr (WJ > 1) {
        double *red = reinterpret_cast<double *>(smem_raw);     // reuse the ring and the slices: [WJ][7][IB]
        __syncthreads();                                         // every warp is out of both
        if (lq == 0) {
#pragma unroll
            for (int h = 0; h < NH; ++h) {
                const int irow = wi * (32 * NH) + h * 32 + li;
#pragma unroll
                for (int c = 0; c < 7; ++c) red[((size_t)wj * 7 + c) * IB + irow] = out64[h][c];
            }
        }
        __syncthreads();
        if (wj == 0 && lq == 0) {
#pragma unroll
            for (int h = 0; h < NH; ++h) {
                const int irow = wi * (32 * NH) + h * 32 + li;
#pragma unroll
                for (int c = 0; c < 7; ++c) {
                    double ssum = out64[h][c];
                    for (int w = 1; w < WJ; ++w) ssum += red[((size_t)w * 7 + c) * IB + irow];
                    out64[h][c] = ssum;
                }
            }
        }
    }
    if (wj == 0 && lq == 0) {
#pragma unroll
        for (int h = 0; h < NH; ++h) {
            const int slot = blockIdx.x * IB + wi * (32 * NH) + h * 32 + li;    // slot < n_i_pad always
#pragma unroll
            for (int c = 0; c < 7; ++c)
                p.partial[((size_t)(p.split0 + blockIdx.y) * 7 + c) * p.n_i_pad + slot] = out64[h][c];
        }
    }
    TL_STAMP(blockIdx.y * gridDim.x + blockIdx.x, 4);
}

// ------------------------------------------------------------------ a6-a7: finalize
// ONE launch, two roles, grid = (ceil(n_i / 32), 7 + 32), CTA = 32 x W threads:
//   blockIdx.y <  7 : fixed-order sum of the S split partials of quantity q = blockIdx.y for 32
//                     consecutive SLOTS of the (possibly reordered) block -- lanes along i (coalesced
//                     256 B rows), warps along the splits with eight loads in flight each, then the W
//                     warps in order; slot s is active particle k = perm[s] (perm = NULL: k = s).
//   blockIdx.y >= 7 : ONE list row per CTA (k = 32 blockIdx.x + blockIdx.y - 7): nnb / overflow from the
//                     row counter (re-zeroed for the next call) and a bitonic sort of the stored entries
//                     in shared memory by the whole CTA (sortP ints; sortP = 0: rows too long, left in
//                     append order).  Sorting makes the list output deterministic and equal to the
//                     oracle's ascending rows.
template <int W>
__global__ void __launch_bounds__(32 * W) finalize_kernel(int32_t n_i, int32_t n_i_pad, int32_t S, int32_t cap,
                                                          int32_t sortP, const unsigned long long *__restrict__ perm,
                                                          const double *__restrict__ blk_dev,
                                                          const double *__restrict__ partial,
                                                          int32_t *__restrict__ cnt, double *__restrict__ acc,
                                                          double *__restrict__ jerk, double *__restrict__ pot,
                                                          int32_t *__restrict__ nnb, int32_t *__restrict__ nblist,
                                                          int32_t *__restrict__ overflow) {
    extern __shared__ int32_t sbuf[];
    __shared__ double red[W][32];
    __shared__ int32_t row_cnt;
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    TL_STAMP(4096 + blockIdx.y * gridDim.x + blockIdx.x, 0);
    // launched with programmatic stream serialization: the grid is resident before the force kernel
    // has drained; everything it reads is valid after this wait (a no-op in an ordinary launch)
    pdl_wait();
    TL_STAMP(4096 + blockIdx.y * gridDim.x + blockIdx.x, 1);
    {
        double t_unused = 0.0;
        if (!spec_block(blk_dev, n_i, t_unused)) return;
    }
    if (blockIdx.y < 7) {
        const int q = blockIdx.y;
        const int slot = blockIdx.x * 32 + lane;       // slot < n_i_pad always (n_i_pad is a multiple of 32)
        const double *src = partial + (size_t)q * n_i_pad + slot;
        const size_t stride = (size_t)7 * n_i_pad;
        double s = 0.0;
        for (int base = w; base < S; base += 8 * W) {
            double v[8];
#pragma unroll
            for (int u = 0; u < 8; ++u) {
                const int sp = base + u * W;
                v[u] = sp < S ? src[(size_t)sp * stride] : 0.0;
            }
#pragma unroll
            for (int u = 0; u < 8; ++u) s += v[u];
        }
        red[w][lane] = s;
        __syncthreads();
        if (w == 0 && slot < n_i) {
            double t = red[0][lane];
#pragma unroll
            for (int ww = 1; ww < W; ++ww) t += red[ww][lane];
            const int k = perm ? perm_slot(perm, slot) : slot;
            if (q < 3) acc[3 * k + q] = t;
            else if (q < 6) jerk[3 * k + q - 3] = t;
            else pot[k] = -t;
        }
        TL_STAMP(4096 + blockIdx.y * gridDim.x + blockIdx.x, 2);
        return;
    }
    const int k = blockIdx.x * 32 + (blockIdx.y - 7);
    if (k >= n_i) return;
    if (threadIdx.x == 0) {
        const int32_t c0 = cnt[k];
        nnb[k] = c0;
        overflow[k] = c0 > cap ? 1 : 0;
        cnt[k] = 0;     // keep the counters zero between calls
        row_cnt = c0;
    }
    __syncthreads();
    const int c = min(row_cnt, cap);
    if (c < 2 || !nblist || sortP == 0) return;
    int Pk = 32;
    while (Pk < c) Pk <<= 1;                                     // this row's power of two (<= sortP)
    int32_t *row = nblist + (int64_t)k * cap;
    const int T = 32 * W;
    for (int e = threadIdx.x; e < Pk; e += T) sbuf[e] = e < c ? row[e] : 0x7fffffff;
    __syncthreads();
    for (int size = 2; size <= Pk; size <<= 1) {
        for (int stride = size >> 1; stride > 0; stride >>= 1) {
            for (int e = threadIdx.x; e < (Pk >> 1); e += T) {
                const int lo = 2 * e - (e & (stride - 1));       // index with bit `stride` clear
                const int hi = lo + stride;
                const bool up = (lo & size) == 0;
                const int32_t x = sbuf[lo], y = sbuf[hi];
                if ((x > y) == up) { sbuf[lo] = y; sbuf[hi] = x; }
            }
            __syncthreads();
        }
    }
    for (int e = threadIdx.x; e < c; e += T) row[e] = sbuf[e];
    TL_STAMP(4096 + blockIdx.y * gridDim.x + blockIdx.x, 3);
}

// ------------------------------------------------------------------ NEXT-2: neighbour (irregular) force
// For each active i: predict i and every listed neighbour j to time t from the FP64 j-state ("predict
// all neighbours and do the force calculation within one loop") and sum the neighbour forces
// ("the irregular force accumulates only the neighbor forces"), all in FP64.  One warp per i;
// lanes stride over the list row (one 128 B line of the AoS copy per neighbour: gather-bound); the
// seven sums are reduced with a fixed xor-shuffle tree.
struct BodyD { double m, x[3], v[3]; };
// The body of a 128 B state line (seven 16 B pieces q0..q6) predicted to time t.
__device__ __forceinline__ BodyD predict_line(double2 q0, double2 q1, double2 q2, double2 q3, double2 q4, double2 q5, double2 q6,
                                              double t) {
    const double x[3] = {q0.y, q1.x, q1.y}, v[3] = {q2.x, q2.y, q3.x}, a[3] = {q3.y, q4.x, q4.y};
    const double jk[3] = {q5.x, q5.y, q6.x};
    const double dt = t - q6.y, c2 = taylor_c2(dt), c3 = taylor_c3(dt);
    BodyD b;
    b.m = q0.x;
#pragma unroll
    for (int c = 0; c < 3; ++c) predict_component(x[c], v[c], a[c], jk[c], dt, c2, c3, b.x[c], b.v[c]);
    return b;
}
// One 256-bit load (sm_100: LDG.E.256), 32 B-aligned.  A scattered gather is bound by the tag look-ups of L1, one per
// lane and instruction: half as many instructions per record, half as many look-ups.  An ORDINARY global load, not
// the read-only (.nc) path: the state lines and predicted records it fetches are rewritten by the kernels ahead in
// the same programmatic chain (correctors, predict64_kernel), and only ordinary loads are ordered after
// griddepcontrol.wait by construction rather than by where they happen to stand in the source.
__device__ __forceinline__ void ld256(const double *p, double &a, double &b, double &c, double &d) {
    asm volatile("ld.global.v4.f64 {%0, %1, %2, %3}, [%4];" : "=d"(a), "=d"(b), "=d"(c), "=d"(d) : "l"(p));
}
__device__ __forceinline__ BodyD predict_body(const double *__restrict__ aos, int32_t j, double t) {
    const double *p = aos + (int64_t)j * AOS_D;
    double2 q0, q1, q2, q3, q4, q5, q6, q7;
    ld256(p, q0.x, q0.y, q1.x, q1.y); ld256(p + 4, q2.x, q2.y, q3.x, q3.y);
    ld256(p + 8, q4.x, q4.y, q5.x, q5.y); ld256(p + 12, q6.x, q6.y, q7.x, q7.y);
    return predict_line(q0, q1, q2, q3, q4, q5, q6, t);
}

// Large blocks (NB_TUNE_IRR_PRED_MIN): every body is predicted ONCE to the block time into a 64 B record
// {m, x[3], v[3], pad} -- the values predict_body returns, bit for bit -- and the neighbour loop gathers those
// records instead of predicting each listed neighbour again from its 128 B state line: half the gathered bytes
// and no Taylor polynomial per pair.  Pays once the block's lists hold more lines than the one pass over all N
// moves (~10^4 bodies at 150 neighbours).
constexpr int P64_D = 8;
__global__ void __launch_bounds__(256) predict64_kernel(int64_t N, double t, const double *__restrict__ aos,
                                                        double *__restrict__ p64) {
    const int64_t j = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= N) return;
    const BodyD b = predict_body(aos, (int32_t)j, t);
    double2 *o = reinterpret_cast<double2 *>(p64 + j * P64_D);
    o[0] = make_double2(b.m, b.x[0]); o[1] = make_double2(b.x[1], b.x[2]);
    o[2] = make_double2(b.v[0], b.v[1]); o[3] = make_double2(b.v[2], 0.0);
}
// The predicted body j at time t: from its record (PRED) or from its state line.
template <bool PRED>
__device__ __forceinline__ BodyD body_at(const double *__restrict__ src, int32_t j, double t) {
    if constexpr (PRED) {
        const double *p = src + (int64_t)j * P64_D;
        BodyD b;
        double pad;
        ld256(p, b.m, b.x[0], b.x[1], b.x[2]);
        ld256(p + 4, b.v[0], b.v[1], b.v[2], pad);
        return b;
    } else {
        return predict_body(src, j, t);
    }
}

// ACCUM: add to acc / jerk / pot instead of overwriting them (nb_block_step: regular + irregular = total).
// PRED: `aos` is the array of predicted records (predict64_kernel) instead of the state lines.
// idx_i = NULL: the identity block.  rows_by_body / out_by_body: the list rows (and nnb) / the outputs are
// indexed by BODY (the persistent lists and scratch of the two-level AC stepping) instead of by k.
template <bool ACCUM, bool PRED = false>
__global__ void __launch_bounds__(256) irregular_kernel(int32_t n_i, int32_t cap, double t,
                                                        const double *__restrict__ blk_dev,
                                                        int32_t rows_by_body, int32_t out_by_body,
                                                        const int32_t *__restrict__ idx_i,
                                                        const int32_t *__restrict__ nnb,
                                                        const int32_t *__restrict__ nblist,
                                                        const double *__restrict__ aos, double *__restrict__ acc,
                                                        double *__restrict__ jerk, double *__restrict__ pot) {
    const int lane = threadIdx.x & 31;
    const int k = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    pdl_wait();
    // (a speculative launch: the index is requested together with the descriptor; n_i is still the launch's capacity
    // here, which the host keeps <= N, the size of the list buffer)
    const int32_t i_spec = (blk_dev && idx_i && k < n_i) ? idx_i[k] : 0;
    if (!spec_block(blk_dev, n_i, t)) return;
    if (k >= n_i) return;
    const int32_t i = blk_dev && idx_i ? i_spec : idx_i ? idx_i[k] : k;
    const BodyD I = body_at<PRED>(aos, i, t);
    const int64_t kr = rows_by_body ? i : k, ko = out_by_body ? i : k;
    const int cnt = min(nnb[kr], cap);
    const int32_t *row = nblist + kr * cap;
    double s[7];
#pragma unroll
    for (int q = 0; q < 7; ++q) s[q] = 0.0;
    // State lines: the 32 neighbours of a batch are fetched COOPERATIVELY -- eight lanes read the 16 B pieces of one
    // 128 B line (one tag look-up in L1 per neighbour instead of seven: the scattered 16 B loads of a lane-per-line
    // gather kept the L1 tag stage 94 % busy), the lines go through a warp-private slice of shared memory, and every
    // lane then takes ITS neighbour (entry e0 + lane, as a lane-strided loop would: same terms, same order of the
    // sums).  Predicted records (64 B: two 256-bit loads per lane) gain nothing from it (measured; nor do 256-bit loads
    // help the cooperative fetch) and keep the direct gather; so do
    // tiny blocks (<= COOP_MIN bodies: latency matters there, not throughput, and the direct gather is a shorter chain).
    constexpr int PIECES = 8, STRIDE = PIECES + 1;               // (stride 144 B: the LDS.128 of a quarter-warp hit distinct banks)
    constexpr int COOP_MIN = 64;
    __shared__ double2 sbuf[PRED ? 1 : 8][PRED ? 1 : 32 * STRIDE];
    double2 *wb = sbuf[PRED ? 0 : threadIdx.x >> 5];
    const double2 *src2 = reinterpret_cast<const double2 *>(aos);
    for (int e0 = 0; e0 < cnt; e0 += 32) {
        const int32_t j = e0 + lane < cnt ? row[e0 + lane] : -1;
        BodyD J;
        if (PRED || n_i <= COOP_MIN) {                           // (uniform over the grid)
            if (j < 0 || j == i) continue;                       // (past the end; a list never holds its owner: be safe)
            J = body_at<PRED>(aos, j, t);
        } else {
            double2 pc[PIECES];
#pragma unroll
            for (int r = 0; r < PIECES; ++r) {                   // straight-line: the eight loads are in flight together
                const int32_t js = __shfl_sync(0xffffffffu, j, r * (32 / PIECES) + lane / PIECES);
                pc[r] = src2[(int64_t)(js >= 0 ? js : i) * (AOS_D / 2) + (lane % PIECES)];     // (past the end: any valid line)
            }
#pragma unroll
            for (int r = 0; r < PIECES; ++r) wb[(r * (32 / PIECES) + lane / PIECES) * STRIDE + lane % PIECES] = pc[r];
            __syncwarp();
            if (j >= 0 && j != i) {
                const double2 *q = wb + lane * STRIDE;
                J = predict_line(q[0], q[1], q[2], q[3], q[4], q[5], q[6], t);
            }
            __syncwarp();
            if (j < 0 || j == i) continue;
        }
        const double dx = J.x[0] - I.x[0], dy = J.x[1] - I.x[1], dz = J.x[2] - I.x[2];
        const double dvx = J.v[0] - I.v[0], dvy = J.v[1] - I.v[1], dvz = J.v[2] - I.v[2];
        const double r2 = fma(dz, dz, fma(dy, dy, dx * dx));
        const double rv = fma(dz, dvz, fma(dy, dvy, dx * dvx));
        const double rinv = rsqrt(r2);
        const double rinv2 = rinv * rinv;
        const double mrinv = J.m * rinv;
        const double mrinv3 = mrinv * rinv2;
        const double alpha = -3.0 * rv * rinv2;
        s[0] = fma(mrinv3, dx, s[0]); s[1] = fma(mrinv3, dy, s[1]); s[2] = fma(mrinv3, dz, s[2]);
        s[3] = fma(mrinv3, fma(alpha, dx, dvx), s[3]);
        s[4] = fma(mrinv3, fma(alpha, dy, dvy), s[4]);
        s[5] = fma(mrinv3, fma(alpha, dz, dvz), s[5]);
        s[6] -= mrinv;
    }
#pragma unroll
    for (int off = 16; off > 0; off >>= 1)
#pragma unroll
        for (int q = 0; q < 7; ++q) s[q] += __shfl_xor_sync(0xffffffffu, s[q], off);
    if (lane == 0) {
        if (ACCUM) {
#pragma unroll
            for (int q = 0; q < 3; ++q) { acc[3 * ko + q] += s[q]; jerk[3 * ko + q] += s[3 + q]; }
            if (pot) pot[ko] += s[6];
        } else {
            acc[3 * ko + 0] = s[0]; acc[3 * ko + 1] = s[1]; acc[3 * ko + 2] = s[2];
            jerk[3 * ko + 0] = s[3]; jerk[3 * ko + 1] = s[4]; jerk[3 * ko + 2] = s[5];
            if (pot) pot[ko] = s[6];
        }
    }
}

// ------------------------------------------------------------------ NEXT-3: block selection, corrector, steps
// Block selection (P:47 block time steps; section 3.3.1).  The paper keeps an index list sorted by
// step so that a CPU never scans N particles; on this chip a scan of t0 + dt over N = 1M bodies is
// 16 MB of HBM traffic (~3 us), so the selection is the definition itself in three small launches:
// t_next = min_j (t0_j + dt_j); per-CTA counts of {j : t0_j + dt_j == t_next}; ordered scatter.
constexpr int SEL_CHUNK = 2048;      // bodies per CTA of the count / scatter kernels
__device__ __forceinline__ unsigned long long ordered_key(double x) {      // monotone map double -> uint64
    const unsigned long long b = (unsigned long long)__double_as_longlong(x);
    return (b >> 63) ? ~b : (b | 0x8000000000000000ull);
}
__device__ __forceinline__ double key_to_double(unsigned long long k) {
    const unsigned long long b = (k >> 63) ? (k & 0x7fffffffffffffffull) : ~k;
    return __longlong_as_double((long long)b);
}

__global__ void __launch_bounds__(256) next_time_kernel(int64_t N, const double *__restrict__ t0,
                                                        const double *__restrict__ dtj,
                                                        unsigned long long *__restrict__ tmin_key) {
    unsigned long long best = ~0ull;
    for (int64_t j = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; j < N; j += (int64_t)gridDim.x * blockDim.x)
        best = min(best, ordered_key(t0[j] + dtj[j]));
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) best = min(best, __shfl_xor_sync(0xffffffffu, best, off));
    __shared__ unsigned long long wbest[8];
    if ((threadIdx.x & 31) == 0) wbest[threadIdx.x >> 5] = best;
    __syncthreads();
    if (threadIdx.x == 0) {
#pragma unroll
        for (int w = 1; w < 8; ++w) best = min(best, wbest[w]);
        atomicMin(tmin_key, best);      // integer atomic: order-independent, reproducible
    }
}

// PASS 0: counts[b] = number of active bodies in chunk b.  PASS 1: chunk b's offset = sum of the counts
// before it (every CTA sums them itself: <= N / 2048 integers), then an ordered ballot compaction, so
// idx_act is ascending.  The last CTA of pass 1 also writes the total and t_next to result[0..1].
template <int PASS>
__global__ void __launch_bounds__(256) select_active_kernel(int64_t N, const double *__restrict__ t0,
                                                            const double *__restrict__ dtj,
                                                            const unsigned long long *__restrict__ tmin_key,
                                                            int32_t *__restrict__ counts,
                                                            int32_t *__restrict__ idx_act,
                                                            double *__restrict__ result) {
    const double tn = key_to_double(*tmin_key);
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    __shared__ int32_t wsum[8];
    __shared__ int32_t base_s;
    int32_t base = 0;
    if (PASS == 1) {
        int32_t part = 0;
        for (int b = threadIdx.x; b < (int)blockIdx.x; b += 256) part += counts[b];
#pragma unroll
        for (int off = 16; off > 0; off >>= 1) part += __shfl_xor_sync(0xffffffffu, part, off);
        if (lane == 0) wsum[w] = part;
        __syncthreads();
        if (threadIdx.x == 0) {
            int32_t tsum = 0;
#pragma unroll
            for (int q = 0; q < 8; ++q) tsum += wsum[q];
            base_s = tsum;
        }
        __syncthreads();
        base = base_s;
        __syncthreads();
    }
    const int64_t cbeg = (int64_t)blockIdx.x * SEL_CHUNK;
    int32_t running = 0;                                    // active bodies of this chunk before the current slab
    for (int s = 0; s < SEL_CHUNK; s += 256) {
        const int64_t j = cbeg + s + threadIdx.x;
        const bool act = j < N && (t0[j] + dtj[j] == tn);
        const unsigned bal = __ballot_sync(0xffffffffu, act);
        if (lane == 0) wsum[w] = __popc(bal);
        __syncthreads();
        int32_t before = 0, slab = 0;
#pragma unroll
        for (int q = 0; q < 8; ++q) {
            const int32_t cq = wsum[q];
            before += q < w ? cq : 0;
            slab += cq;
        }
        if (PASS == 1 && act) idx_act[base + running + before + __popc(bal & ((1u << lane) - 1u))] = (int32_t)j;
        running += slab;
        __syncthreads();
    }
    if (threadIdx.x == 0) {
        if (PASS == 0) counts[blockIdx.x] = running;
        if (PASS == 1 && blockIdx.x == gridDim.x - 1) {
            result[0] = tn;
            result[1] = (double)(base + running);
        }
    }
}

// The selection of the block loop (nb_block_step / nb_ac_step and their loops): TWO ordinary launches, no grid-wide
// synchronisation.  (1) select_min_kernel: t_next = min_j (t0_j + dt_j) into `key` (~0 on entry; the other slot is
// reset for the next call).  (2) select_scatter_kernel: one CTA per 2048-body chunk counts its active bodies,
// publishes the count tagged with this call's epoch, sums the counts of the chunks before it as they appear
// (decoupled look-back: lower chunks are scheduled first and never wait for higher ones) and writes its bodies
// in ascending order; the last chunk writes the block descriptor {t_next, n, n_regular, status} to device memory
// and to the host's ring.  TWO (two-level AC stepping): the active bodies whose REGULAR step is due as well
// (tR_j + dtR_j == t_next) are also listed, ascending, in idx_reg.
// A BATCH of blocks is enqueued without the host in between: once a block needs the host (too large for the
// speculative chain, a regular step due, past t_stop) `*stall` is set and every later selection of the batch does
// nothing, so that block's lists stay in place.  (The flag is written by an EARLIER kernel only.)
__global__ void __launch_bounds__(256) select_min_kernel(int64_t N, const double *__restrict__ t0,
                                                         const double *__restrict__ dtj, unsigned long long *key,
                                                         unsigned long long *key_next, const int32_t *stall,
                                                         double *__restrict__ ring) {
    pdl_wait();
    if (*stall) {
        if (blockIdx.x == 0 && threadIdx.x == 0) {
            *key_next = ~0ull;
            *reinterpret_cast<volatile double *>(ring + 3) = (double)BLK_SKIPPED;
        }
        return;
    }
    unsigned long long best = ~0ull;
    for (int64_t j = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; j < N; j += (int64_t)gridDim.x * blockDim.x)
        best = min(best, ordered_key(t0[j] + dtj[j]));
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) best = min(best, __shfl_xor_sync(0xffffffffu, best, off));
    __shared__ unsigned long long wbest[8];
    if ((threadIdx.x & 31) == 0) wbest[threadIdx.x >> 5] = best;
    __syncthreads();
    if (threadIdx.x == 0) {
#pragma unroll
        for (int w = 1; w < 8; ++w) best = min(best, wbest[w]);
        atomicMin(key, best);
        if (blockIdx.x == 0) *key_next = ~0ull;
    }
}

// The same minimum from per-chunk minima (section 3.3.1: the search for the due particles must not cost O(N)
// per block when the deep blocks hold a handful of particles).  cmin[b] = min over chunk b of t0 + dt, kept
// between blocks; the correctors flag the chunks of the bodies they integrate (dirty[b] = 1) and only those
// chunks are scanned again here.  One CTA per chunk; everything else reads one word.  The library flags every
// chunk when the state or the steps are replaced from outside the chain.
__global__ void __launch_bounds__(256) select_min_chunks_kernel(int64_t N, const double *__restrict__ t0,
                                                                const double *__restrict__ dtj,
                                                                unsigned long long *__restrict__ cmin,
                                                                int32_t *__restrict__ dirty, unsigned long long *key,
                                                                unsigned long long *key_next, const int32_t *stall,
                                                                double *__restrict__ ring) {
    pdl_wait();
    const int b = blockIdx.x;
    // (the three words the decision rests on are requested together: one trip to L2, not three in a row)
    const int32_t stalled = *stall, is_dirty = dirty[b];
    const unsigned long long old_min = cmin[b];
    if (stalled) {
        if (blockIdx.x == 0 && threadIdx.x == 0) {
            *key_next = ~0ull;
            *reinterpret_cast<volatile double *>(ring + 3) = (double)BLK_SKIPPED;
        }
        return;
    }
    if (!is_dirty) {                                  // (uniform over the CTA)
        if (threadIdx.x == 0) {
            atomicMin(key, old_min);
            if (b == 0) *key_next = ~0ull;
        }
        return;
    }
    unsigned long long best = ~0ull;
#pragma unroll
    for (int u = 0; u < SEL_CHUNK / 256; ++u) {
        const int64_t j = (int64_t)b * SEL_CHUNK + u * 256 + threadIdx.x;
        if (j < N) best = min(best, ordered_key(t0[j] + dtj[j]));
    }
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) best = min(best, __shfl_xor_sync(0xffffffffu, best, off));
    __shared__ unsigned long long wbest[8];
    if ((threadIdx.x & 31) == 0) wbest[threadIdx.x >> 5] = best;
    __syncthreads();
    if (threadIdx.x == 0) {
#pragma unroll
        for (int w = 1; w < 8; ++w) best = min(best, wbest[w]);
        cmin[b] = best;
        dirty[b] = 0;
        atomicMin(key, best);
        if (b == 0) *key_next = ~0ull;
    }
}

template <bool TWO>
__global__ void __launch_bounds__(256) select_scatter_kernel(int64_t N, const double *__restrict__ t0,
                                                             const double *__restrict__ dtj, const unsigned long long *key,
                                                             unsigned long long *pub, uint32_t epoch,
                                                             int32_t *__restrict__ idx_act, double *__restrict__ result,
                                                             const double *__restrict__ tR, const double *__restrict__ dtR,
                                                             int32_t *__restrict__ idx_reg, double t_stop, int32_t spec_cap,
                                                             int32_t *stall, double *__restrict__ ring,
                                                             const unsigned long long *__restrict__ cmin, int32_t nchunk) {
    pdl_wait();
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    // (requested together: one trip to L2)
    const int32_t stalled = *stall;
    const unsigned long long kmin = *key;
    unsigned long long my_min = cmin ? cmin[blockIdx.x] : 0ull;
    if (stalled) return;
    constexpr int PER = SEL_CHUNK / 256;
    __shared__ int32_t wsum[8], wsum2[8];
    __shared__ int32_t base_s, base2_s;
    const double tn = key_to_double(kmin);
    // The look-back below waits for the chunks before this one.  That is safe because the host caps the grid at the
    // number of CTAs the device holds at once (blk_setup) and a CTA takes its chunks in ascending order: every chunk
    // somebody waits for belongs to a CTA that is resident or will be as soon as kernels AHEAD of this one drain --
    // never to one queued behind a spinning CTA.  (Up to that cap -- 2.4M bodies on a B200 -- the grid is one CTA
    // per chunk, as before.)
    for (int b = blockIdx.x; b < nchunk; b += gridDim.x) {
    if (b != (int)blockIdx.x) {
        __syncthreads();                            // the shared words of the previous chunk are done with
        my_min = cmin ? cmin[b] : 0ull;
    }
    const bool here = !cmin || my_min == kmin;      // only a chunk whose own minimum is t_next holds due bodies
    // ---- this chunk's active bodies (kept as flags) and their number
    bool act[PER], due[PER];
    int32_t cntc = 0, cnt2 = 0;
#pragma unroll
    for (int u = 0; u < PER; ++u) {
        const int64_t j = (int64_t)b * SEL_CHUNK + u * 256 + threadIdx.x;
        act[u] = here && j < N && (t0[j] + dtj[j] == tn);
        due[u] = TWO && act[u] && (tR[j] + dtR[j] == tn);
        cntc += act[u] ? 1 : 0;
        cnt2 += due[u] ? 1 : 0;
    }
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) {
        cntc += __shfl_xor_sync(0xffffffffu, cntc, off);
        cnt2 += __shfl_xor_sync(0xffffffffu, cnt2, off);
    }
    if (lane == 0) { wsum[w] = cntc; wsum2[w] = cnt2; }
    __syncthreads();
    int32_t mine = 0, mine2 = 0;
#pragma unroll
    for (int q = 0; q < 8; ++q) { mine += wsum[q]; mine2 += wsum2[q]; }
    if (threadIdx.x == 0)       // publish: epoch (32 bits) | regular count (16 bits) | count (16 bits); a chunk holds <= 2048
        atomicExch(pub + b, ((unsigned long long)epoch << 32) | ((unsigned long long)mine2 << 16) | (unsigned long long)mine);
    // ---- look-back: the counts of all chunks before this one, as they appear
    int32_t part = 0, part2 = 0;
    for (int q = threadIdx.x; q < b; q += 256) {
        unsigned long long v;
        do { v = *reinterpret_cast<volatile unsigned long long *>(pub + q); } while ((uint32_t)(v >> 32) != epoch);
        part += (int32_t)(v & 0xffffu);
        part2 += (int32_t)((v >> 16) & 0xffffu);
    }
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) {
        part += __shfl_xor_sync(0xffffffffu, part, off);
        part2 += __shfl_xor_sync(0xffffffffu, part2, off);
    }
    __syncthreads();
    if (lane == 0) { wsum[w] = part; wsum2[w] = part2; }
    __syncthreads();
    if (threadIdx.x == 0) {
        int32_t tsum = 0, tsum2 = 0;
#pragma unroll
        for (int q = 0; q < 8; ++q) { tsum += wsum[q]; tsum2 += wsum2[q]; }
        base_s = tsum; base2_s = tsum2;
    }
    __syncthreads();
    int32_t running = base_s, running2 = base2_s;
    // ---- ordered compaction (ascending indices)
    if (mine > 0) {
#pragma unroll
        for (int u = 0; u < PER; ++u) {
            const int64_t j = (int64_t)b * SEL_CHUNK + u * 256 + threadIdx.x;
            const unsigned bal = __ballot_sync(0xffffffffu, act[u]);
            const unsigned bal2 = __ballot_sync(0xffffffffu, due[u]);
            __syncthreads();
            if (lane == 0) { wsum[w] = __popc(bal); wsum2[w] = __popc(bal2); }
            __syncthreads();
            int32_t before = 0, slab = 0, before2 = 0, slab2 = 0;
#pragma unroll
            for (int q = 0; q < 8; ++q) {
                const int32_t cq = wsum[q], cq2 = wsum2[q];
                before += q < w ? cq : 0;
                slab += cq;
                before2 += q < w ? cq2 : 0;
                slab2 += cq2;
            }
            if (act[u]) idx_act[running + before + __popc(bal & ((1u << lane) - 1u))] = (int32_t)j;
            if (due[u]) idx_reg[running2 + before2 + __popc(bal2 & ((1u << lane) - 1u))] = (int32_t)j;
            running += slab;
            running2 += slab2;
        }
    }
    if (b == nchunk - 1 && threadIdx.x == 0) {
        const int32_t n1 = base_s + mine, n2 = base2_s + mine2;
        // spec_cap = 0: no speculative chain follows.  TWO: that chain cannot take a regular step.
        const int status = tn > t_stop ? BLK_PAST_T_STOP
                           : (n1 > 0 && n1 <= spec_cap && n2 == 0) ? BLK_SPECULATIVE : BLK_NEEDS_HOST;
        result[0] = tn; result[1] = (double)n1; result[2] = (double)n2; result[3] = (double)status;
        if (status != BLK_SPECULATIVE) *stall = 1;
        volatile double *rv = ring;      // mapped host memory: the status word last, after the rest is visible system-wide
        rv[0] = tn; rv[1] = (double)n1; rv[2] = (double)n2;
        __threadfence_system();
        rv[3] = (double)status;
    }
    }       // chunks of this CTA
}

constexpr double DT_MIN_FACTOR = 1.0 / 1099511627776.0;     // 2^-40: no step below dt_max 2^-40 (reading R32)
// Largest power of two not above x (x > 0, normal): clear the mantissa.
__device__ __forceinline__ double pow2_floor(double x) {
    return __longlong_as_double(__double_as_longlong(x) & 0x7ff0000000000000ll);
}
__device__ __forceinline__ double norm3(const double *a) { return sqrt(fma(a[2], a[2], fma(a[1], a[1], a[0] * a[0]))); }

// Start-up steps (textbook: dt = eta_s |a| / |j|, quantised to a power of 0.5, <= dt_max).
__global__ void __launch_bounds__(256) init_steps_kernel(int64_t N, int64_t Ns, double eta_s, double dt_max,
                                                         const double *__restrict__ soa, double *__restrict__ dtj) {
    const int64_t j = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= N) return;
    double a[3], jk[3];
#pragma unroll
    for (int c = 0; c < 3; ++c) { a[c] = soa[(7 + c) * Ns + j]; jk[c] = soa[(10 + c) * Ns + j]; }
    double req = eta_s * norm3(a) / norm3(jk);
    if (req != req) req = dt_max;                                   // |a| = |j| = 0: nothing known (reading R32)
    dtj[j] = pow2_floor(fmin(fmax(req, dt_max * DT_MIN_FACTOR), dt_max));
}

// Fourth-order Hermite corrector + new block step for the n active bodies (Makino & Aarseth 1992):
// the acceleration over the step is the cubic Hermite interpolant of (a0, j0) at t0 and (a1, j1) at
// t1 = t0 + dt; its second and third derivatives a2, a3 extend the predictor's Taylor series by the
// dt^4, dt^5 (x) and dt^3, dt^4 (v) terms.  New step: Aarseth's criterion with the derivatives at t1,
// then the block rule (double once if allowed and t1 is commensurate, else halve while too long).
// One thread per active body; reads its 128 B line of the gather copy, writes both copies.  FP64.
__global__ void __launch_bounds__(128) correct_kernel(int32_t n, int64_t Ns, double t1, double eta, double dt_max,
                                                      const double *__restrict__ blk_dev,
                                                      const int32_t *__restrict__ idx,
                                                      const double *__restrict__ acc1,
                                                      const double *__restrict__ jerk1, double *__restrict__ soa,
                                                      double *__restrict__ aos, double *__restrict__ dtj,
                                                      int32_t *__restrict__ sel_dirty) {
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    pdl_wait();
    const int32_t i_spec = (blk_dev && k < n) ? idx[k] : 0;    // (requested together with the descriptor; n: the launch's capacity)
    if (!spec_block(blk_dev, n, t1)) return;
    if (k >= n) return;
    const int64_t i = blk_dev ? i_spec : idx[k];
    const double2 *p = reinterpret_cast<const double2 *>(aos + i * AOS_D);
    const double2 q0 = p[0], q1 = p[1], q2 = p[2], q3 = p[3], q4 = p[4], q5 = p[5], q6 = p[6];
    const double m = q0.x;
    const double x0[3] = {q0.y, q1.x, q1.y}, v0[3] = {q2.x, q2.y, q3.x}, a0[3] = {q3.y, q4.x, q4.y};
    const double j0[3] = {q5.x, q5.y, q6.x};
    const double h = dtj[i];                       // = t1 - t0 for an active body
    const double h2 = h * h, h3 = h2 * h, h4 = h2 * h2, h5 = h4 * h;
    double x1[3], v1[3], a1[3], j1[3], a2e[3], a3[3];
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        a1[c] = acc1[3 * k + c];
        j1[c] = jerk1[3 * k + c];
        const double da = a0[c] - a1[c];
        const double a2 = (-6.0 * da - h * (4.0 * j0[c] + 2.0 * j1[c])) / h2;
        a3[c] = (12.0 * da + 6.0 * h * (j0[c] + j1[c])) / h3;
        x1[c] = x0[c] + v0[c] * h + a0[c] * h2 / 2.0 + j0[c] * h3 / 6.0 + a2 * h4 / 24.0 + a3[c] * h5 / 120.0;
        v1[c] = v0[c] + a0[c] * h + j0[c] * h2 / 2.0 + a2 * h3 / 6.0 + a3[c] * h4 / 24.0;
        a2e[c] = a2 + h * a3[c];                   // second derivative at the end of the step
    }
    const double na = norm3(a1), nj = norm3(j1), n2 = norm3(a2e), n3 = norm3(a3);
    const double req = sqrt(eta * (na * n2 + nj * nj) / (nj * n3 + n2 * n2));
    double d = h;
    if (req > 0.0) {        // req = 0 or NaN carries no information: the step is kept (reading R32)
        const double d2 = 2.0 * d, ratio = t1 / d2, dmin = dt_max * DT_MIN_FACTOR;
        if (req >= d2 && d2 <= dt_max && ratio == floor(ratio)) d = d2;
        else
            while (d > req && d > dmin) d *= 0.5;
    }
    store_body(i, Ns, m, x1, v1, a1, j1, t1, soa, aos);
    dtj[i] = d;
    if (sel_dirty) sel_dirty[i / SEL_CHUNK] = 1;      // this chunk's minimum of t0 + dt is out of date (select_min_chunks_kernel)
}

// ------------------------------------------------------------------ NEXT-3: two-level Ahmad-Cohen stepping
// (regular force from outside the neighbour radius on large steps, irregular force from the neighbours on
// small steps, the regular force and its first derivative extrapolated in between; readings R33-R38.)
struct AcState {
    double *aI, *jI, *aR, *jR;        // [N][3] irregular force at t0 over the body's list; regular force at tR
    double *tR, *dtR;                 // [N] last regular time, regular step (the irregular step is dtj)
    int32_t *nnb, *list;              // [N], [N][cap] the body's neighbour list (from its last regular step)
};
__device__ __forceinline__ double aarseth_req(const double *a, const double *j, const double *a2e, const double *a3,
                                              double eta) {
    const double na = norm3(a), nj = norm3(j), n2 = norm3(a2e), n3 = norm3(a3);
    return sqrt(eta * (na * n2 + nj * nj) / (nj * n3 + n2 * n2));
}
// Block rule (readings R29, R32): candidate d; doubled once if allowed, else halved while above req.
__device__ __forceinline__ double block_rule(double req, double d, double t1, double dt_max) {
    if (req > 0.0) {
        const double d2 = 2.0 * d, ratio = t1 / d2, dmin = dt_max * DT_MIN_FACTOR;
        if (req >= d2 && d2 <= dt_max && ratio == floor(ratio)) d = d2;
        else
            while (d > req && d > dmin) d *= 0.5;
    }
    return d;
}

// Start-up (R37): forces are in place (aR, jR, lists from the full regular pass; aI, jI over those lists);
// writes the total a0, j0 into the stored state and the two steps; counts overflowed lists (R38).
__global__ void __launch_bounds__(128) ac_start_kernel(int64_t N, int64_t Ns, int32_t cap, double t_start, double eta_s,
                                                       double dt_max, const AcState A, double *__restrict__ soa,
                                                       double *__restrict__ aos, double *__restrict__ dtj,
                                                       int32_t *__restrict__ n_overflow) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    const double2 *p = reinterpret_cast<const double2 *>(aos + i * AOS_D);
    const double2 q0 = p[0], q1 = p[1], q2 = p[2], q3 = p[3];
    const double x0[3] = {q0.y, q1.x, q1.y}, v0[3] = {q2.x, q2.y, q3.x};
    double aI[3], jI[3], aR[3], jR[3], a0[3], j0[3];
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        aI[c] = A.aI[3 * i + c]; jI[c] = A.jI[3 * i + c]; aR[c] = A.aR[3 * i + c]; jR[c] = A.jR[3 * i + c];
        a0[c] = aI[c] + aR[c]; j0[c] = jI[c] + jR[c];
    }
    auto init_step = [&](const double *a, const double *j) {
        double req = eta_s * norm3(a) / norm3(j);
        if (req != req) req = dt_max;
        return pow2_floor(fmin(fmax(req, dt_max * DT_MIN_FACTOR), dt_max));
    };
    const double dR = init_step(aR, jR);
    const int32_t nn = A.nnb[i];
    const double dI = nn == 0 ? dR : fmin(init_step(aI, jI), dR);
    if (nn > cap) atomicAdd(n_overflow, 1);
    store_body(i, Ns, q0.x, x0, v0, a0, j0, t_start, soa, aos);
    A.tR[i] = t_start; A.dtR[i] = dR; dtj[i] = dI;
}

// Both correctors for the n irregular-active bodies idx[0..n) at time t (R34, R35).  aIo / jIo: irregular
// force over the OLD list, indexed by body.  A body whose regular step is due as well (tR + dtR == t) finds
// its slot r in the ascending idx_reg[0..n_reg) and there the new-list forces: regular rg_acc/rg_jerk[r],
// irregular in_acc/in_jerk[r], new count rg_nnb[r] (rows are copied by ac_store_rows_kernel afterwards).
__global__ void __launch_bounds__(128) ac_correct_kernel(int32_t n, int64_t Ns, double t, double eta_I, double eta_R,
                                                         double dt_max, const double *__restrict__ blk_dev,
                                                         const int32_t *__restrict__ idx,
                                                         const double *__restrict__ aIo, const double *__restrict__ jIo,
                                                         int32_t n_reg, const int32_t *__restrict__ idx_reg,
                                                         const double *__restrict__ rg_acc, const double *__restrict__ rg_jerk,
                                                         const double *__restrict__ in_acc, const double *__restrict__ in_jerk,
                                                         const int32_t *__restrict__ rg_nnb, const AcState A,
                                                         double *__restrict__ soa, double *__restrict__ aos,
                                                         double *__restrict__ dtj, int32_t *__restrict__ sel_dirty) {
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    pdl_wait();
    const int32_t i_spec = (blk_dev && k < n) ? idx[k] : 0;    // (requested together with the descriptor; n: the launch's capacity <= N)
    if (!spec_block(blk_dev, n, t)) return;
    if (k >= n) return;
    const int64_t i = blk_dev ? i_spec : idx[k];
    const double2 *p = reinterpret_cast<const double2 *>(aos + i * AOS_D);
    const double2 q0 = p[0], q1 = p[1], q2 = p[2], q3 = p[3], q4 = p[4], q5 = p[5], q6 = p[6];
    const double m = q0.x;
    const double x0[3] = {q0.y, q1.x, q1.y}, v0[3] = {q2.x, q2.y, q3.x}, a0[3] = {q3.y, q4.x, q4.y};
    const double j0[3] = {q5.x, q5.y, q6.x};
    const double h = dtj[i];                                   // = t - t0: the irregular step
    const double tR = A.tR[i], hR = A.dtR[i];
    const bool due = tR + hR == t;
    const double h2 = h * h, h3 = h2 * h, h4 = h2 * h2, h5 = h4 * h;
    double x1[3], v1[3], a1[3], j1[3], a2e[3], a3[3], aI1[3], jI1[3], aR0[3], jR0[3];
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        aI1[c] = aIo[3 * i + c]; jI1[c] = jIo[3 * i + c];
        aR0[c] = A.aR[3 * i + c]; jR0[c] = A.jR[3 * i + c];
        a1[c] = aI1[c] + (aR0[c] + jR0[c] * (t - tR));         // regular force extrapolated
        j1[c] = jI1[c] + jR0[c];
        const double da = a0[c] - a1[c];
        const double a2 = (-6.0 * da - h * (4.0 * j0[c] + 2.0 * j1[c])) / h2;
        a3[c] = (12.0 * da + 6.0 * h * (j0[c] + j1[c])) / h3;
        x1[c] = x0[c] + v0[c] * h + a0[c] * h2 / 2.0 + j0[c] * h3 / 6.0 + a2 * h4 / 24.0 + a3[c] * h5 / 120.0;
        v1[c] = v0[c] + a0[c] * h + j0[c] * h2 / 2.0 + a2 * h3 / 6.0 + a3[c] * h4 / 24.0;
        a2e[c] = a2 + h * a3[c];
    }
    double dI, dR = hR;
    int32_t nn = A.nnb[i];
    if (!due) {
        dI = block_rule(aarseth_req(aI1, jI1, a2e, a3, eta_I), h, t, dt_max);
    } else {
        int lo = 0, hi = n_reg - 1;                             // slot of body i in the ascending regular list
        while (lo < hi) {
            const int mid = (lo + hi) >> 1;
            if (idx_reg[mid] < (int32_t)i) lo = mid + 1; else hi = mid;
        }
        const int r = lo;
        const double g2 = hR * hR, g3 = g2 * hR, g4 = g2 * g2, g5 = g4 * hR;
        double aRn[3], jRn[3], aIn[3], jIn[3], a2Re[3], a3R[3];
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            aRn[c] = rg_acc[3 * r + c]; jRn[c] = rg_jerk[3 * r + c];
            aIn[c] = in_acc[3 * r + c]; jIn[c] = in_jerk[3 * r + c];
            const double atot = aRn[c] + aIn[c], jtot = jRn[c] + jIn[c];
            const double aR1 = atot - aI1[c], jR1 = jtot - jI1[c];          // regular force w.r.t. the OLD list
            const double da = aR0[c] - aR1;
            const double a2R = (-6.0 * da - hR * (4.0 * jR0[c] + 2.0 * jR1)) / g2;
            a3R[c] = (12.0 * da + 6.0 * hR * (jR0[c] + jR1)) / g3;
            x1[c] = x1[c] + (a2R * g4 / 24.0 + a3R[c] * g5 / 120.0);       // the regular correction (R35)
            v1[c] = v1[c] + (a2R * g3 / 6.0 + a3R[c] * g4 / 24.0);
            a2Re[c] = a2R + hR * a3R[c];
            a1[c] = atot; j1[c] = jtot;
        }
        dR = block_rule(aarseth_req(aRn, jRn, a2Re, a3R, eta_R), hR, t, dt_max);
        dI = block_rule(aarseth_req(aIn, jIn, a2e, a3, eta_I), h, t, dt_max);
        nn = rg_nnb[r];
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            aI1[c] = aIn[c]; jI1[c] = jIn[c];
            A.aR[3 * i + c] = aRn[c]; A.jR[3 * i + c] = jRn[c];
        }
        A.tR[i] = t; A.dtR[i] = dR; A.nnb[i] = nn;
    }
    dI = nn == 0 ? dR : fmin(dI, dR);                          // R36; never above the regular step
#pragma unroll
    for (int c = 0; c < 3; ++c) { A.aI[3 * i + c] = aI1[c]; A.jI[3 * i + c] = jI1[c]; }
    store_body(i, Ns, m, x1, v1, a1, j1, t, soa, aos);
    dtj[i] = dI;
    if (sel_dirty) sel_dirty[i / SEL_CHUNK] = 1;
}

// New list rows of the regular-active bodies into the persistent by-body lists: one warp per row.
__global__ void __launch_bounds__(256) ac_store_rows_kernel(int32_t n_reg, int32_t cap, const int32_t *__restrict__ idx_reg,
                                                            const int32_t *__restrict__ rg_nnb,
                                                            const int32_t *__restrict__ rg_list, int32_t *__restrict__ list) {
    const int lane = threadIdx.x & 31;
    const int r = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    if (r >= n_reg) return;
    const int64_t i = idx_reg[r];
    const int c = min(rg_nnb[r], cap);
    for (int e = lane; e < c; e += 32) list[i * cap + e] = rg_list[(int64_t)r * cap + e];
}

// block-level overflow count of the regular pass (R38)
__global__ void __launch_bounds__(256) count_overflow_kernel(int32_t n, const int32_t *__restrict__ ovf, int32_t *__restrict__ out) {
    int32_t c = 0;
    for (int k = blockIdx.x * blockDim.x + threadIdx.x; k < n; k += gridDim.x * blockDim.x) c += ovf[k] ? 1 : 0;
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) c += __shfl_xor_sync(0xffffffffu, c, off);
    if ((threadIdx.x & 31) == 0 && c) atomicAdd(out, c);
}

// nb_ac_init's precondition (every body at t_start): number of bodies whose t0 differs
__global__ void __launch_bounds__(256) count_not_at_kernel(int64_t N, const double *__restrict__ t0, double t_start,
                                                           int32_t *__restrict__ out) {
    int32_t c = 0;
    for (int64_t j = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; j < N; j += (int64_t)gridDim.x * blockDim.x)
        c += t0[j] != t_start ? 1 : 0;
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) c += __shfl_xor_sync(0xffffffffu, c, off);
    if ((threadIdx.x & 31) == 0 && c) atomicAdd(out, c);
}
// nb_ac_set_radii: h2_all[idx[k]] = h2[k]; an index outside [0, N) is ignored
__global__ void __launch_bounds__(256) scatter_radii_kernel(int32_t n, int64_t N, const int32_t *__restrict__ idx,
                                                            const double *__restrict__ h2, double *__restrict__ h2_all) {
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= n) return;
    const int64_t j = idx[k];
    if (j >= 0 && j < N) h2_all[j] = h2[k];
}

// Inspection: the FP64 state back in the caller's layout (tests, energy checks, checkpoints).
__global__ void __launch_bounds__(256) export_state_kernel(int64_t N, int64_t Ns, const double *__restrict__ soa,
                                                           const double *__restrict__ dtj, double *__restrict__ m,
                                                           double *__restrict__ x0, double *__restrict__ v0,
                                                           double *__restrict__ a0, double *__restrict__ j0,
                                                           double *__restrict__ t0, double *__restrict__ dt) {
    const int64_t j = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= N) return;
    m[j] = soa[j];
    t0[j] = soa[13 * Ns + j];
    if (dt) dt[j] = dtj[j];
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        x0[3 * j + c] = soa[(1 + c) * Ns + j]; v0[3 * j + c] = soa[(4 + c) * Ns + j];
        a0[3 * j + c] = soa[(7 + c) * Ns + j]; j0[3 * j + c] = soa[(10 + c) * Ns + j];
    }
}

}  // namespace nbreg
