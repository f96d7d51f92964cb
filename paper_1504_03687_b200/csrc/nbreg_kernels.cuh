// nbreg_kernels.cuh -- sm_100a device code of libnbreg (see include/nbreg.h for the contract).
//
//   relayout_kernel   a1  AoS [N][3] FP64 -> internal SoA FP64                    (HBM-bound)
//   predict_kernel    a2  Hermite predictor, FP64 -> predicted record (48 B/body) (HBM-bound)
//   force_kernel      a3-a6  i-block x j-tile pairwise sum + neighbour lists      (FP32 issue-bound)
//   finalize_kernel   a6-a7  fixed-order sum over j-splits, write-back, counters  (tiny)
//
// Predicted record: 80 B per body, five float4 with every value DUPLICATED into an aligned pair,
//   q0 = (xh,xh, yh,yh)  q1 = (zh,zh, m,m)  q2 = (xl,xl, yl,yl)  q3 = (zl,zl, vx,vx)  q4 = (vy,vy, vz,vz)
// so that one warp-uniform LDS.128 hands the force kernel two ready-made f32x2 operands: each thread
// owns a PAIR of i-particles and every FP32 operation of the pair arithmetic is one packed
// FADD2/FMUL2/FFMA2 (sm_100 only) -- half the issue slots of scalar FP32 at the same lane rate.
// x = hi + lo with hi = fl32(x), lo = fl32(x - hi): positions carry 48 significant bits, so
// (hi_j - hi_i) + (lo_j - lo_i) is the FP64 difference rounded once to FP32 -- the pair arithmetic
// after that is plain FP32.  A j-tile (256 records, 20 KB) is ONE TMA bulk copy.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace nbreg {

constexpr int TJ = 256;        // j-particles per shared-memory tile
constexpr int RECQ = 5;        // float4 per predicted record (80 B)
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
__device__ __forceinline__ void fence_proxy_async_smem() {   // generic-proxy accesses before, async-proxy (TMA) after
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
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
// xp = x0 + v0 dt + a0 dt^2/2 + j0 dt^3/6,  vp = v0 + a0 dt + j0 dt^2/2   (reading R2)
__global__ void __launch_bounds__(256) predict_kernel(int64_t N, int64_t Npad, int64_t Ns, double t,
                                                      const double *__restrict__ soa, float4 *__restrict__ rec) {
    int64_t j = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= Npad) return;
    float4 *r = rec + j * RECQ;
    if (j >= N) {   // ghost padding: massless, far away, never a neighbour, contributes exactly 0
        r[0] = make_float4(GHOST_POS, GHOST_POS, GHOST_POS, GHOST_POS);
        r[1] = make_float4(GHOST_POS, GHOST_POS, 0.f, 0.f);
        r[2] = r[3] = r[4] = make_float4(0.f, 0.f, 0.f, 0.f);
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
    const float mf = __double2float_rn(soa[j]);
    r[0] = make_float4(hi[0], hi[0], hi[1], hi[1]);
    r[1] = make_float4(hi[2], hi[2], mf, mf);
    r[2] = make_float4(lo[0], lo[0], lo[1], lo[1]);
    r[3] = make_float4(lo[2], lo[2], vf[0], vf[0]);
    r[4] = make_float4(vf[1], vf[1], vf[2], vf[2]);
}

__global__ void __launch_bounds__(256) unpack_predicted_kernel(int64_t N, const float4 *__restrict__ rec,
                                                               double *__restrict__ xp, double *__restrict__ vp) {
    int64_t j = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= N) return;
    const float4 *r = rec + j * RECQ;
    const float4 q0 = r[0], q1 = r[1], q2 = r[2], q3 = r[3], q4 = r[4];
    xp[3 * j + 0] = (double)q0.x + (double)q2.x;
    xp[3 * j + 1] = (double)q0.z + (double)q2.z;
    xp[3 * j + 2] = (double)q1.x + (double)q3.x;
    vp[3 * j + 0] = (double)q3.z;
    vp[3 * j + 1] = (double)q4.x;
    vp[3 * j + 2] = (double)q4.z;
}

// ------------------------------------------------------------------ a3-a6: force kernel
struct ForceParams {
    const float4 *rec;            // predicted records, Npad x RECQ
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

// Two active particles (lane halves .x / .y) held in registers, NEGATED so that every difference is
// one packed add:  d = j + (-i).
struct IPair {
    float2 nxh, nyh, nzh, nxl, nyl, nzl, nvx, nvy, nvz, h2;
};

__device__ __forceinline__ float2 lo2(const float4 &q) { return make_float2(q.x, q.y); }
__device__ __forceinline__ float2 hi2(const float4 &q) { return make_float2(q.z, q.w); }

// r^2 of one (i, j) pair in SCALAR FP32, operation for operation what the packed fast path does per
// half (IEEE round-to-nearest either way), so both paths classify a pair identically.
__device__ __forceinline__ float scalar_r2(float nxh, float nyh, float nzh, float nxl, float nyl, float nzl,
                                           const float4 &q0, const float4 &q1, const float4 &q2, const float4 &q3) {
    const float dx = __fadd_rn(__fadd_rn(q0.x, nxh), __fadd_rn(q2.x, nxl));
    const float dy = __fadd_rn(__fadd_rn(q0.z, nyh), __fadd_rn(q2.z, nyl));
    const float dz = __fadd_rn(__fadd_rn(q1.x, nzh), __fadd_rn(q3.x, nzl));
    return __fmaf_rn(dz, dz, __fmaf_rn(dy, dy, __fmul_rn(dx, dx)));
}

// Rare path: some lane saw r2 < h2 inside the last group of j's.  Lanes of one warp hold DIFFERENT i,
// so the vote only gates the path; each flagged lane re-scans the group for each of its two particles
// and takes one slot of that particle's row with an integer atomic (rows are shared with the other
// j-splits and warps).
__device__ __noinline__ void append_neighbours(float nxh, float nyh, float nzh, float nxl, float nyl, float nzl,
                                               float h2, int32_t my_idx, int32_t k, const float4 *trec,
                                               int32_t jglob0, int32_t cap, int32_t *cnt, int32_t *nblist) {
    for (int u = 0; u < UNROLL_J; ++u) {
        const float4 *r = trec + u * RECQ;
        const float r2 = scalar_r2(nxh, nyh, nzh, nxl, nyl, nzl, r[0], r[1], r[2], r[3]);
        const int32_t jg = jglob0 + u;
        if (r2 < h2 && jg != my_idx) {
            const int32_t pos = atomicAdd(cnt + k, 1);
            if (pos < cap) nblist[(int64_t)k * cap + pos] = jg;
        }
    }
}

// Each thread owns one PAIR of i-particles; WI warps along i (64 i each), WJ warps along j (each takes
// TJ/WJ j's of every tile).  CTA = 32*WI*WJ threads, i-block = 64*WI.
template <int WI, int WJ, int MINB>
__global__ void __launch_bounds__(32 * WI *WJ, MINB) force_kernel(const ForceParams p) {
    constexpr int NW = WI * WJ;
    constexpr int IB = 64 * WI;
    constexpr int SUB = TJ / WJ;
    constexpr uint32_t TILE_BYTES = TJ * RECQ * sizeof(float4);
    static_assert(SUB % UNROLL_J == 0, "sub-tile must be a multiple of the group");

    extern __shared__ __align__(128) unsigned char smem_raw[];
    float4 *srec = reinterpret_cast<float4 *>(smem_raw);                       // [NSTAGE][TJ][RECQ]
    uint64_t *full = reinterpret_cast<uint64_t *>(smem_raw + (size_t)NSTAGE * TILE_BYTES);
    int *done = reinterpret_cast<int *>(full + NSTAGE);                        // warps finished with a stage

    const int tid = threadIdx.x;
    const int warp = tid >> 5, lane = tid & 31;
    const int wi = warp % WI, wj = warp / WI;

    const int tile_begin = blockIdx.y * p.tiles_per_split;
    const int tile_end = min(tile_begin + p.tiles_per_split, p.ntiles);
    const int ntile = max(tile_end - tile_begin, 0);

    // ---- a3: gather the i-state (the i-particle IS predicted record idx_i[k]; reading R3)
    IPair I;
    int32_t my_idx[2], my_k[2];
    {
        float v[2][10];
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            const int k = blockIdx.x * IB + wi * 64 + h * 32 + lane;
            my_k[h] = k;
            if (k < p.n_i) {
                const int32_t idx = p.idx_i[k];
                const float4 *r = p.rec + (size_t)idx * RECQ;
                const float4 q0 = r[0], q1 = r[1], q2 = r[2], q3 = r[3], q4 = r[4];
                my_idx[h] = idx;
                v[h][0] = -q0.x; v[h][1] = -q0.z; v[h][2] = -q1.x;
                v[h][3] = -q2.x; v[h][4] = -q2.z; v[h][5] = -q3.x;
                v[h][6] = -q3.z; v[h][7] = -q4.x; v[h][8] = -q4.z;
                v[h][9] = fmaxf(__double2float_rn(p.h2_i[k]), TINY_H2);
            } else {    // padding lane: far from everything (also from the ghost j's), result discarded
                my_idx[h] = -1;
                v[h][0] = v[h][1] = v[h][2] = GHOST_POS;        // i.e. position -GHOST_POS
                v[h][3] = v[h][4] = v[h][5] = v[h][6] = v[h][7] = v[h][8] = 0.f;
                v[h][9] = TINY_H2;
            }
        }
        I.nxh = make_float2(v[0][0], v[1][0]); I.nyh = make_float2(v[0][1], v[1][1]);
        I.nzh = make_float2(v[0][2], v[1][2]); I.nxl = make_float2(v[0][3], v[1][3]);
        I.nyl = make_float2(v[0][4], v[1][4]); I.nzl = make_float2(v[0][5], v[1][5]);
        I.nvx = make_float2(v[0][6], v[1][6]); I.nvy = make_float2(v[0][7], v[1][7]);
        I.nvz = make_float2(v[0][8], v[1][8]); I.h2 = make_float2(v[0][9], v[1][9]);
    }

    if (tid == 0) {
#pragma unroll
        for (int s = 0; s < NSTAGE; ++s) {
            mbar_init(&full[s], 1);
            done[s] = 0;
        }
        fence_mbar_init();
    }
    __syncthreads();

    auto issue = [&](int tile, int s) {     // one bulk copy per tile (20 KB), completion on full[s]
        mbar_arrive_expect_tx(&full[s], TILE_BYTES);
        bulk_g2s(srec + (size_t)s * TJ * RECQ, p.rec + (size_t)tile * TJ * RECQ, TILE_BYTES, &full[s]);
    };
    if (tid == 0) {
        for (int s = 0; s < NSTAGE && s < ntile; ++s) issue(tile_begin + s, s);
    }

    double acc64[2][7];
#pragma unroll
    for (int h = 0; h < 2; ++h)
#pragma unroll
        for (int q = 0; q < 7; ++q) acc64[h][q] = 0.0;

    const float2 m3 = make_float2(-3.0f, -3.0f);

    for (int it = 0; it < ntile; ++it) {
        const int s = it % NSTAGE;
        mbar_wait(&full[s], (uint32_t)((it / NSTAGE) & 1));
        const float4 *trec = srec + ((size_t)s * TJ + wj * SUB) * RECQ;
        const int32_t jbase = (tile_begin + it) * TJ + wj * SUB;

        float2 ax = make_float2(0.f, 0.f), ay = ax, az = ax, jx = ax, jy = ax, jz = ax, ph = ax;

#pragma unroll 1
        for (int g = 0; g < SUB; g += UNROLL_J) {
            bool hit = false;
#pragma unroll
            for (int u = 0; u < UNROLL_J; ++u) {
                const float4 *r = trec + (g + u) * RECQ;      // warp-uniform addresses: LDS.128 broadcasts
                const float4 q0 = r[0], q1 = r[1], q2 = r[2], q3 = r[3], q4 = r[4];
                const float2 dx = __fadd2_rn(__fadd2_rn(lo2(q0), I.nxh), __fadd2_rn(lo2(q2), I.nxl));
                const float2 dy = __fadd2_rn(__fadd2_rn(hi2(q0), I.nyh), __fadd2_rn(hi2(q2), I.nyl));
                const float2 dz = __fadd2_rn(__fadd2_rn(lo2(q1), I.nzh), __fadd2_rn(lo2(q3), I.nzl));
                const float2 dvx = __fadd2_rn(hi2(q3), I.nvx);
                const float2 dvy = __fadd2_rn(lo2(q4), I.nvy);
                const float2 dvz = __fadd2_rn(hi2(q4), I.nvz);
                const float2 r2 = __ffma2_rn(dz, dz, __ffma2_rn(dy, dy, __fmul2_rn(dx, dx)));
                const float2 rv = __ffma2_rn(dz, dvz, __ffma2_rn(dy, dvy, __fmul2_rn(dx, dvx)));
                const bool nb0 = r2.x < I.h2.x, nb1 = r2.y < I.h2.y;   // neighbour (or the self pair, r2 == 0)
                hit |= nb0 | nb1;
                float2 rinv;
                rinv.x = nb0 ? 0.f : rsqrt_sfu(r2.x);       // masked before any product: no inf * 0
                rinv.y = nb1 ? 0.f : rsqrt_sfu(r2.y);
                const float2 rinv2 = __fmul2_rn(rinv, rinv);
                const float2 mrinv = __fmul2_rn(hi2(q1), rinv);
                const float2 mrinv3 = __fmul2_rn(mrinv, rinv2);
                const float2 alpha = __fmul2_rn(__fmul2_rn(rv, rinv2), m3);
                ph = __fadd2_rn(ph, mrinv);
                ax = __ffma2_rn(mrinv3, dx, ax);
                ay = __ffma2_rn(mrinv3, dy, ay);
                az = __ffma2_rn(mrinv3, dz, az);
                jx = __ffma2_rn(mrinv3, __ffma2_rn(alpha, dx, dvx), jx);
                jy = __ffma2_rn(mrinv3, __ffma2_rn(alpha, dy, dvy), jy);
                jz = __ffma2_rn(mrinv3, __ffma2_rn(alpha, dz, dvz), jz);
            }
            if (__any_sync(0xffffffffu, hit)) {     // ~1 % of groups at N_b ~ 150, N = 1M
                if (hit) {
                    const float4 *tg = trec + g * RECQ;
                    append_neighbours(I.nxh.x, I.nyh.x, I.nzh.x, I.nxl.x, I.nyl.x, I.nzl.x, I.h2.x, my_idx[0], my_k[0],
                                      tg, jbase + g, p.cap, p.cnt, p.nblist);
                    append_neighbours(I.nxh.y, I.nyh.y, I.nzh.y, I.nxl.y, I.nyl.y, I.nzl.y, I.h2.y, my_idx[1], my_k[1],
                                      tg, jbase + g, p.cap, p.cnt, p.nblist);
                }
            }
        }
        // tile flush: FP32 partial sums of <= SUB terms go into the FP64 running sums
        acc64[0][0] += (double)ax.x; acc64[1][0] += (double)ax.y;
        acc64[0][1] += (double)ay.x; acc64[1][1] += (double)ay.y;
        acc64[0][2] += (double)az.x; acc64[1][2] += (double)az.y;
        acc64[0][3] += (double)jx.x; acc64[1][3] += (double)jx.y;
        acc64[0][4] += (double)jy.x; acc64[1][4] += (double)jy.y;
        acc64[0][5] += (double)jz.x; acc64[1][5] += (double)jz.y;
        acc64[0][6] += (double)ph.x; acc64[1][6] += (double)ph.y;

        // Stage hand-back without a CTA barrier: the LAST warp to finish with stage s refills it, so
        // warps drift up to NSTAGE-1 tiles apart instead of meeting at a __syncthreads every tile.
        __syncwarp();
        if (lane == 0) {
            __threadfence_block();                       // my reads of stage s are done (release)
            if (atomicAdd(&done[s], 1) == NW - 1) {
                done[s] = 0;
                __threadfence_block();
                if (it + NSTAGE < ntile) {
                    fence_proxy_async_smem();            // generic reads -> async-proxy overwrite
                    issue(tile_begin + it + NSTAGE, s);
                }
            }
        }
    }

    // ---- a6: fixed-order reduction over the WJ warps that shared these i, then one partial per split
    if constexpr (WJ > 1) {
        double *red = reinterpret_cast<double *>(smem_raw);     // reuse the tile ring: [WJ][7][IB]
        __syncthreads();                                         // every warp is out of the ring
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            const int il = wi * 64 + h * 32 + lane;
#pragma unroll
            for (int q = 0; q < 7; ++q) red[((size_t)wj * 7 + q) * IB + il] = acc64[h][q];
        }
        __syncthreads();
        if (wj == 0) {
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                const int il = wi * 64 + h * 32 + lane;
#pragma unroll
                for (int q = 0; q < 7; ++q) {
                    double ssum = acc64[h][q];
                    for (int w = 1; w < WJ; ++w) ssum += red[((size_t)w * 7 + q) * IB + il];
                    acc64[h][q] = ssum;
                }
            }
        }
    }
    if (wj == 0) {
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            const int k = my_k[h];    // k < n_i_pad always
#pragma unroll
            for (int q = 0; q < 7; ++q)
                p.partial[((size_t)blockIdx.y * 7 + q) * p.n_i_pad + k] = acc64[h][q];
        }
    }
}

// ------------------------------------------------------------------ a6-a7: finalize
// One warp per active particle: lanes stride over the S split partials (fixed assignment), then a
// fixed-order shuffle tree -- deterministic, and S loads in flight instead of a serial chain.
__global__ void __launch_bounds__(256) finalize_kernel(int32_t n_i, int32_t n_i_pad, int32_t S, int32_t cap,
                                                       const double *__restrict__ partial, int32_t *__restrict__ cnt,
                                                       double *__restrict__ acc, double *__restrict__ jerk,
                                                       double *__restrict__ pot, int32_t *__restrict__ nnb,
                                                       int32_t *__restrict__ overflow) {
    const int lane = threadIdx.x & 31;
    const int k = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    if (k >= n_i) return;
    double s[7];
#pragma unroll
    for (int q = 0; q < 7; ++q) s[q] = 0.0;
    for (int sp = lane; sp < S; sp += 32) {
#pragma unroll
        for (int q = 0; q < 7; ++q) s[q] += partial[((size_t)sp * 7 + q) * n_i_pad + k];
    }
#pragma unroll
    for (int off = 16; off > 0; off >>= 1)
#pragma unroll
        for (int q = 0; q < 7; ++q) s[q] += __shfl_down_sync(0xffffffffu, s[q], off);
    if (lane == 0) {
        acc[3 * k + 0] = s[0]; acc[3 * k + 1] = s[1]; acc[3 * k + 2] = s[2];
        jerk[3 * k + 0] = s[3]; jerk[3 * k + 1] = s[4]; jerk[3 * k + 2] = s[5];
        pot[k] = -s[6];
        const int32_t c = cnt[k];
        nnb[k] = c;
        overflow[k] = c > cap ? 1 : 0;
        cnt[k] = 0;     // keep the counters zero between calls
    }
}

}  // namespace nbreg
