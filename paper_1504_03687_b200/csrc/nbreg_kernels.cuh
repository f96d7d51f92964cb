// nbreg_kernels.cuh -- sm_100a device code of libnbreg (see include/nbreg.h for the contract).
//
//   relayout_kernel   a1  AoS [N][3] FP64 -> internal SoA FP64                    (HBM-bound)
//   predict_kernel    a2  Hermite predictor, FP64 -> predicted record (48 B/body) (HBM-bound)
//   force_kernel      a3-a6  i-block x j-tile pairwise sum + neighbour lists      (FP32 issue-bound)
//   finalize_kernel   a6-a7  fixed-order sum over j-splits, write-back, counters  (tiny)
//
// Predicted record (three float4 streams so that a j-tile is three 1-D bulk copies):
//   pA[j] = (x_hi, y_hi, z_hi, m)    pB[j] = (x_lo, y_lo, z_lo, 0)    pC[j] = (vx, vy, vz, 0)
// with x = hi + lo, hi = fl32(x), lo = fl32(x - hi): positions carry 48 significant bits, so
// (hi_j - hi_i) + (lo_j - lo_i) is the FP64 difference rounded once to FP32 -- the pair
// arithmetic after that is plain FP32.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace nbreg {

constexpr int TJ = 256;        // j-particles per shared-memory tile
constexpr int NSTAGE = 3;      // tiles in flight per CTA (bulk-copy ring)
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
__device__ __forceinline__ float rsqrt_sfu(float x) {   // one MUFU.RSQ, no denormal fix-up code
    float y;
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

// ------------------------------------------------------------------ a1: re-layout
// in: m[N], x0[N][3], v0[N][3], a0[N][3], j0[N][3], t0[N]  ->  soa[14][Ns] (component-major).
__global__ void __launch_bounds__(256) relayout_kernel(int64_t N, int64_t Ns, const double *__restrict__ m,
                                                       const double *__restrict__ x0, const double *__restrict__ v0,
                                                       const double *__restrict__ a0, const double *__restrict__ j0,
                                                       const double *__restrict__ t0, double *__restrict__ soa) {
    int64_t j = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= N) return;
    soa[0 * Ns + j] = m[j];
    soa[13 * Ns + j] = t0[j];
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        soa[(1 + c) * Ns + j] = x0[3 * j + c];
        soa[(4 + c) * Ns + j] = v0[3 * j + c];
        soa[(7 + c) * Ns + j] = a0[3 * j + c];
        soa[(10 + c) * Ns + j] = j0[3 * j + c];
    }
}

// ------------------------------------------------------------------ a2: predictor
// xp = x0 + dt (v0 + dt (a0/2 + dt j0/6)),  vp = v0 + dt (a0 + dt j0/2)   (reading R2)
__global__ void __launch_bounds__(256) predict_kernel(int64_t N, int64_t Npad, int64_t Ns, double t,
                                                      const double *__restrict__ soa, float4 *__restrict__ pA,
                                                      float4 *__restrict__ pB, float4 *__restrict__ pC) {
    int64_t j = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= Npad) return;
    if (j >= N) {   // ghost padding: massless, far away, never a neighbour, contributes exactly 0
        pA[j] = make_float4(GHOST_POS, GHOST_POS, GHOST_POS, 0.f);
        pB[j] = make_float4(0.f, 0.f, 0.f, 0.f);
        pC[j] = make_float4(0.f, 0.f, 0.f, 0.f);
        return;
    }
    const double dt = t - soa[13 * Ns + j];
    const double c2 = 0.5 * (dt * dt);                    // dt^2/2: exact for dyadic dt
    const double c3 = (dt * dt * dt) * (1.0 / 6.0);       // dt^3/6: the only inexact coefficient
    float hi[3], lo[3], vf[3];
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const double x = soa[(1 + c) * Ns + j], v = soa[(4 + c) * Ns + j];
        const double a = soa[(7 + c) * Ns + j], jk = soa[(10 + c) * Ns + j];
        // The jerk term is rounded on its own (not fused) so that for dyadic inputs with j0 = 6 q the
        // product rounds back to q dt^3 exactly and the whole sum is exact (tests: bitwise vs oracle).
        const double p3 = __dmul_rn(jk, c3);
        const double xp = __dadd_rn(fma(a, c2, fma(v, dt, x)), p3);
        const double vp = fma(jk, c2, fma(a, dt, v));
        hi[c] = __double2float_rn(xp);
        lo[c] = __double2float_rn(xp - (double)hi[c]);
        vf[c] = __double2float_rn(vp);
    }
    pA[j] = make_float4(hi[0], hi[1], hi[2], __double2float_rn(soa[j]));
    pB[j] = make_float4(lo[0], lo[1], lo[2], 0.f);
    pC[j] = make_float4(vf[0], vf[1], vf[2], 0.f);
}

__global__ void __launch_bounds__(256) unpack_predicted_kernel(int64_t N, const float4 *__restrict__ pA,
                                                               const float4 *__restrict__ pB,
                                                               const float4 *__restrict__ pC, double *__restrict__ xp,
                                                               double *__restrict__ vp) {
    int64_t j = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= N) return;
    const float4 A = pA[j], B = pB[j], C = pC[j];
    xp[3 * j + 0] = (double)A.x + (double)B.x;
    xp[3 * j + 1] = (double)A.y + (double)B.y;
    xp[3 * j + 2] = (double)A.z + (double)B.z;
    vp[3 * j + 0] = (double)C.x;
    vp[3 * j + 1] = (double)C.y;
    vp[3 * j + 2] = (double)C.z;
}

// ------------------------------------------------------------------ a3-a6: force kernel
struct ForceParams {
    const float4 *pA, *pB, *pC;   // predicted records, Npad entries
    const int32_t *idx_i;         // [n_i]
    const double *h2_i;           // [n_i]
    int32_t n_i;
    int32_t n_i_pad;              // n_i rounded up to the CTA's i-block
    int32_t ntiles;               // Npad / TJ
    int32_t tiles_per_split;      // contiguous tiles per blockIdx.y
    int32_t cap;
    int32_t *cnt;                 // [>= n_i] neighbour counters, zero on entry (finalize re-zeroes)
    int32_t *nblist;              // caller's [n_i][cap]
    double *partial;              // [S][7][n_i_pad]
};

struct IState {     // one active particle held in registers
    float xh, yh, zh, xl, yl, zl, vx, vy, vz, h2;
};

__device__ __forceinline__ float pair_r2(const IState &I, const float4 &A, const float4 &B, float &dx, float &dy,
                                         float &dz) {
    // FP64-accurate difference from the hi/lo split; explicit intrinsics so that the fast path and the
    // neighbour slow path get bit-identical r2 (no contraction differences).
    dx = __fadd_rn(__fsub_rn(A.x, I.xh), __fsub_rn(B.x, I.xl));
    dy = __fadd_rn(__fsub_rn(A.y, I.yh), __fsub_rn(B.y, I.yl));
    dz = __fadd_rn(__fsub_rn(A.z, I.zh), __fsub_rn(B.z, I.zl));
    return __fmaf_rn(dz, dz, __fmaf_rn(dy, dy, __fmul_rn(dx, dx)));
}

// Rare path: some lane saw r2 < h2 inside the last group of j's.  Lanes that did re-scan the group
// and append to their own row.  Lanes of one warp hold DIFFERENT i, so the ballot picks the lanes and
// each takes one slot of its own row with an integer atomic (rows are shared with the other j-splits).
__device__ __noinline__ void append_neighbours(const IState I, int32_t my_idx, int32_t k, const float4 *tA,
                                               const float4 *tB, int32_t jglob0, int32_t ngroup, int32_t cap,
                                               int32_t *cnt, int32_t *nblist) {
    for (int u = 0; u < ngroup; ++u) {
        float dx, dy, dz;
        const float r2 = pair_r2(I, tA[u], tB[u], dx, dy, dz);
        const int32_t jg = jglob0 + u;
        if (r2 < I.h2 && jg != my_idx) {
            const int32_t pos = atomicAdd(cnt + k, 1);
            if (pos < cap) nblist[(int64_t)k * cap + pos] = jg;
        }
    }
}

// IT i-particles per thread, WI warps along i, WJ warps along j (each takes TJ/WJ j's of every tile).
template <int IT, int WI, int WJ, int MINB>
__global__ void __launch_bounds__(32 * WI *WJ, MINB) force_kernel(const ForceParams p) {
    constexpr int NT = 32 * WI * WJ;
    constexpr int IB = 32 * IT * WI;
    constexpr int SUB = TJ / WJ;
    static_assert(SUB % UNROLL_J == 0, "sub-tile must be a multiple of the group");

    extern __shared__ __align__(128) unsigned char smem_raw[];
    float4 *sA = reinterpret_cast<float4 *>(smem_raw);            // [NSTAGE][3][TJ]
    uint64_t *full = reinterpret_cast<uint64_t *>(smem_raw + (size_t)NSTAGE * 3 * TJ * sizeof(float4));

    const int tid = threadIdx.x;
    const int warp = tid >> 5, lane = tid & 31;
    const int wi = warp % WI, wj = warp / WI;

    const int tile_begin = blockIdx.y * p.tiles_per_split;
    const int tile_end = min(tile_begin + p.tiles_per_split, p.ntiles);
    const int ntile = max(tile_end - tile_begin, 0);

    // ---- a3: gather the i-state (the i-particle IS predicted record idx_i[k]; reading R3)
    IState I[IT];
    int32_t my_idx[IT], my_k[IT];
#pragma unroll
    for (int t = 0; t < IT; ++t) {
        const int k = blockIdx.x * IB + wi * (32 * IT) + t * 32 + lane;
        my_k[t] = k;
        if (k < p.n_i) {
            const int32_t idx = p.idx_i[k];
            const float4 A = p.pA[idx], B = p.pB[idx], C = p.pC[idx];
            my_idx[t] = idx;
            I[t].xh = A.x; I[t].yh = A.y; I[t].zh = A.z;
            I[t].xl = B.x; I[t].yl = B.y; I[t].zl = B.z;
            I[t].vx = C.x; I[t].vy = C.y; I[t].vz = C.z;
            I[t].h2 = fmaxf(__double2float_rn(p.h2_i[k]), TINY_H2);
        } else {    // padding lane: far from everything (also from the ghost j's), result discarded
            my_idx[t] = -1;
            I[t].xh = I[t].yh = I[t].zh = -GHOST_POS;
            I[t].xl = I[t].yl = I[t].zl = 0.f;
            I[t].vx = I[t].vy = I[t].vz = 0.f;
            I[t].h2 = TINY_H2;
        }
    }

    if (tid == 0) {
#pragma unroll
        for (int s = 0; s < NSTAGE; ++s) mbar_init(&full[s], 1);
        fence_mbar_init();
    }
    __syncthreads();

    auto issue = [&](int tile, int s) {
        float4 *dst = sA + (size_t)s * 3 * TJ;
        const size_t off = (size_t)tile * TJ;
        mbar_arrive_expect_tx(&full[s], 3u * TJ * sizeof(float4));
        bulk_g2s(dst, p.pA + off, TJ * sizeof(float4), &full[s]);
        bulk_g2s(dst + TJ, p.pB + off, TJ * sizeof(float4), &full[s]);
        bulk_g2s(dst + 2 * TJ, p.pC + off, TJ * sizeof(float4), &full[s]);
    };
    if (tid == 0) {
        for (int s = 0; s < NSTAGE && s < ntile; ++s) issue(tile_begin + s, s);
    }

    double acc64[IT][7];
#pragma unroll
    for (int t = 0; t < IT; ++t)
#pragma unroll
        for (int q = 0; q < 7; ++q) acc64[t][q] = 0.0;

    for (int it = 0; it < ntile; ++it) {
        const int s = it % NSTAGE;
        mbar_wait(&full[s], (uint32_t)((it / NSTAGE) & 1));
        const float4 *tA = sA + (size_t)s * 3 * TJ + wj * SUB;
        const float4 *tB = tA + TJ;
        const float4 *tC = tA + 2 * TJ;
        const int32_t jbase = (tile_begin + it) * TJ + wj * SUB;

        float ax[IT], ay[IT], az[IT], jx[IT], jy[IT], jz[IT], ph[IT];
#pragma unroll
        for (int t = 0; t < IT; ++t) ax[t] = ay[t] = az[t] = jx[t] = jy[t] = jz[t] = ph[t] = 0.f;

#pragma unroll 1
        for (int g = 0; g < SUB; g += UNROLL_J) {
            bool hit[IT];
#pragma unroll
            for (int t = 0; t < IT; ++t) hit[t] = false;
#pragma unroll
            for (int u = 0; u < UNROLL_J; ++u) {
                const float4 A = tA[g + u], B = tB[g + u], C = tC[g + u];   // warp-uniform: LDS broadcast
#pragma unroll
                for (int t = 0; t < IT; ++t) {
                    float dx, dy, dz;
                    const float r2 = pair_r2(I[t], A, B, dx, dy, dz);
                    const float dvx = C.x - I[t].vx, dvy = C.y - I[t].vy, dvz = C.z - I[t].vz;
                    const float rv = fmaf(dz, dvz, fmaf(dy, dvy, dx * dvx));
                    const bool nb = r2 < I[t].h2;           // neighbour (or the self pair, r2 == 0)
                    hit[t] |= nb;
                    float rinv = rsqrt_sfu(r2);
                    rinv = nb ? 0.f : rinv;                 // masked before any product: no inf * 0
                    const float rinv2 = rinv * rinv;
                    const float mrinv = A.w * rinv;
                    const float mrinv3 = mrinv * rinv2;
                    const float alpha = (rv * rinv2) * -3.0f;
                    ph[t] += mrinv;
                    ax[t] = fmaf(mrinv3, dx, ax[t]);
                    ay[t] = fmaf(mrinv3, dy, ay[t]);
                    az[t] = fmaf(mrinv3, dz, az[t]);
                    jx[t] = fmaf(mrinv3, fmaf(alpha, dx, dvx), jx[t]);
                    jy[t] = fmaf(mrinv3, fmaf(alpha, dy, dvy), jy[t]);
                    jz[t] = fmaf(mrinv3, fmaf(alpha, dz, dvz), jz[t]);
                }
            }
            bool anyhit = false;
#pragma unroll
            for (int t = 0; t < IT; ++t) anyhit |= hit[t];
            if (__any_sync(0xffffffffu, anyhit)) {     // ~0.5 % of groups at N_b ~ 150, N = 1M
#pragma unroll
                for (int t = 0; t < IT; ++t)
                    if (hit[t])
                        append_neighbours(I[t], my_idx[t], my_k[t], tA + g, tB + g, jbase + g, UNROLL_J, p.cap,
                                          p.cnt, p.nblist);
            }
        }
        // tile flush: FP32 partial sums of <= SUB terms go into the FP64 running sums
#pragma unroll
        for (int t = 0; t < IT; ++t) {
            acc64[t][0] += (double)ax[t]; acc64[t][1] += (double)ay[t]; acc64[t][2] += (double)az[t];
            acc64[t][3] += (double)jx[t]; acc64[t][4] += (double)jy[t]; acc64[t][5] += (double)jz[t];
            acc64[t][6] += (double)ph[t];
        }
        __syncthreads();    // every warp is done with stage s
        if (tid == 0 && it + NSTAGE < ntile) issue(tile_begin + it + NSTAGE, s);
    }

    // ---- a6: fixed-order reduction over the WJ warps that shared these i, then one partial per split
    double *red = reinterpret_cast<double *>(smem_raw);     // reuse the tile ring: [WJ][7][IB]
    if constexpr (WJ > 1) {
        __syncthreads();
#pragma unroll
        for (int t = 0; t < IT; ++t) {
            const int il = wi * (32 * IT) + t * 32 + lane;
#pragma unroll
            for (int q = 0; q < 7; ++q) red[((size_t)wj * 7 + q) * IB + il] = acc64[t][q];
        }
        __syncthreads();
        if (wj == 0) {
#pragma unroll
            for (int t = 0; t < IT; ++t) {
                const int il = wi * (32 * IT) + t * 32 + lane;
#pragma unroll
                for (int q = 0; q < 7; ++q) {
                    double ssum = acc64[t][q];
                    for (int w = 1; w < WJ; ++w) ssum += red[((size_t)w * 7 + q) * IB + il];
                    acc64[t][q] = ssum;
                }
            }
        }
    }
    if (wj == 0) {
#pragma unroll
        for (int t = 0; t < IT; ++t) {
            const int k = my_k[t];    // k < n_i_pad always
#pragma unroll
            for (int q = 0; q < 7; ++q)
                p.partial[((size_t)blockIdx.y * 7 + q) * p.n_i_pad + k] = acc64[t][q];
        }
    }
    (void)NT;
}

// ------------------------------------------------------------------ a6-a7: finalize
__global__ void __launch_bounds__(256) finalize_kernel(int32_t n_i, int32_t n_i_pad, int32_t S, int32_t cap,
                                                       const double *__restrict__ partial, int32_t *__restrict__ cnt,
                                                       double *__restrict__ acc, double *__restrict__ jerk,
                                                       double *__restrict__ pot, int32_t *__restrict__ nnb,
                                                       int32_t *__restrict__ overflow) {
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= n_i) return;
    double s[7];
#pragma unroll
    for (int q = 0; q < 7; ++q) s[q] = 0.0;
    for (int sp = 0; sp < S; ++sp) {        // fixed order: bitwise reproducible
#pragma unroll
        for (int q = 0; q < 7; ++q) s[q] += partial[((size_t)sp * 7 + q) * n_i_pad + k];
    }
    acc[3 * k + 0] = s[0]; acc[3 * k + 1] = s[1]; acc[3 * k + 2] = s[2];
    jerk[3 * k + 0] = s[3]; jerk[3 * k + 1] = s[4]; jerk[3 * k + 2] = s[5];
    pot[k] = -s[6];
    const int32_t c = cnt[k];
    nnb[k] = c;
    overflow[k] = c > cap ? 1 : 0;
    cnt[k] = 0;     // keep the counters zero between calls
}

}  // namespace nbreg
