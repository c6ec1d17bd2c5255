// bt_band.cu -- S4a: band back-transformation  Z <- Q2 (sgn o Q_T)  (first of the
// "two stages" of the eigenvector back transformation), SURVEY.md 8(a) row S4a.
//
// Q2 = prod H_{j,k} over the bulge-chasing reflectors (sweep j, step k; rows j+1+kb .. j+kb+b,
// b = 64), generated sweep-major, so Z <- Q2 Z applies them last-generated first.  H_{j,k} and
// H_{j',k'} commute unless their row ranges overlap, which for 0 < j'-j < b happens only for k' = k
// and k' = k-1; hence the valid order used here:
//   passes of P = 32 consecutive sweeps, last pass first; inside a pass the step index k ascending;
//   inside (pass, k) the sweeps descending, grouped GS at a time into compact-WY blocks
//   I - V T V^H (V = GS reflectors, column t shifted down by t rows: a parallelogram).
//
// Kernel design (one persistent kernel for the whole phase, no GEMM launches):
//  * A work unit is (pass, slab of 64 eigenvector columns).  Every column is independent, so a
//    warp owns 8 columns for the whole unit and keeps its 96-row window of Z IN REGISTERS, in the
//    accumulator layout of mma.sync.m8n8k4.f64 with the roles transposed (m = column of Z,
//    n/k = rows or reflectors).  Lane (g, t) holds column g, rows 8p+2t and 8p+2t+1 of every
//    8-row block p.  With that layout the three products of a WY application
//        Y1 = V^H Z (k = rows),  Y = -T Y1 (k = reflectors),  Z += V Y (k = reflectors)
//    chain through registers without any shuffle: the k-permutation "lane t supplies elements
//    2t+h in k-step h" is applied to both operands of each DMMA.
//  * Only the 8x8 blocks of V inside the parallelogram are multiplied (9 row blocks per column
//    block instead of 12): executed/credited flops = 9/8 (+ the small T product).
//  * V (packed, straight from bulge chasing) and -T (prepared per (pass, k)) reach shared memory by
//    1-D bulk async copies (cp.async.bulk, SASS UBLKCP) issued by a producer warp into a 3-stage
//    ring guarded by full/empty mbarriers; the 8 consumer warps never meet at a CTA barrier.
//    Shared-memory leading dimensions are odd (97, 33), which makes both fragment access patterns
//    (row-fastest for V^H Z, column-fastest for V Y) conflict-free for 128-bit loads.
//  * Z rows enter and leave the register window straight from/to global memory: the window slides
//    down by 64 rows per step, so every row of Z is read once and written once per pass.
//  * Units are handed out by an atomic counter in (pass descending, slab) order; (pass, slab)
//    waits for (pass+1, slab) through a per-slab completion counter in global memory.
#include "eigh_internal.h"

namespace eigh {

constexpr int BT_B = 64;            // band width (reflector length)
constexpr int BT_P = 32;            // sweeps per pass
constexpr int BT_WR = BT_B + BT_P;  // window rows (96)
constexpr int BT_NBLK = BT_WR / 8;  // 12 row blocks
constexpr int BT_LDV = BT_WR + 1;   // 97, odd
constexpr int BT_LDT = BT_P + 1;    // 33, odd
constexpr int BT_VS = BT_LDV * BT_P;        // c128 per V stage
constexpr int BT_TS = BT_LDT * BT_P;        // c128 per T stage
constexpr int BT_STAGES = 3;
constexpr int BT_CWARPS = 8;                // consumer warps
constexpr int BT_NT = 32 * (BT_CWARPS + 1); // + producer warp
constexpr int BT_SLAB = 8 * BT_CWARPS;      // 64 columns per unit

struct BtHeader { int j0, k, slab, flags; };   // flags: 1 first step of unit, 2 last step, 4 terminate
constexpr size_t BT_SMEM = (size_t)BT_STAGES * (BT_VS + BT_TS) * sizeof(c128) + BT_STAGES * sizeof(BtHeader) +
                           2 * BT_STAGES * sizeof(uint64_t) + 64;

static inline int64_t bt_npass(int64_t N) { return N >= 2 ? ceil_div(N - 1, BT_P) : 0; }

size_t bt_tneg_bytes(int64_t N) {
    // stages = sum over passes of ceil((N-1-j0)/64)  <=  npass * kmax
    int64_t st = 0;
    for (int64_t p = 0; p < bt_npass(N); ++p) st += ceil_div(N - 1 - p * BT_P, BT_B);
    return (size_t)st * BT_TS * sizeof(c128) + 256;
}
size_t bt_scratch_bytes(const eigh_handle_s* h) {
    // pass offsets + unit counter + per-slab completion counters + S4b's Y
    const size_t y = (size_t)h->b * h->nev * sizeof(c128);
    return y + (size_t)(bt_npass(h->N) + 8) * sizeof(int64_t) + (size_t)(ceil_div(h->nev, BT_SLAB) + 64) * sizeof(int) + 8192;
}

// ------------------------------------------------------------------ small kernels
// Z[r, c] = sgn[r] * Qt[r + c*ldq]
__global__ void bt_expand_kernel(const double* __restrict__ Qt, int64_t ldq, const double* __restrict__ sgn, int N,
                                 int nev, c128* __restrict__ Z, int64_t ldz) {
    const int c = blockIdx.y;
    const int r = blockIdx.x * blockDim.x + threadIdx.x;
    if (r < N && c < nev) Z[r + (int64_t)c * ldz] = cmake(sgn[r] * Qt[r + (int64_t)c * ldq], 0.0);
}

// pass_off[p] = number of (pass, k) stages of passes < p
__global__ void bt_pass_off_kernel(int N, int npass, int64_t* __restrict__ pass_off) {
    if (threadIdx.x == 0 && blockIdx.x == 0) {
        int64_t s = 0;
        for (int p = 0; p < npass; ++p) {
            pass_off[p] = s;
            s += (N - 1 - p * BT_P + BT_B - 1) / BT_B;
        }
        pass_off[npass] = s;
    }
}

// One CTA per (k = blockIdx.x, pass = blockIdx.y): -T of the GS-sized compact-WY blocks of the 32
// reflectors (sweeps j0..j0+31, step k), written in the padded shared-memory layout of the sweeper
// (Tn[out + in*33]; zero outside the diagonal GS x GS blocks and for reflectors that do not exist).
//   T[j,j] = tau_j,  T[i,j] = -tau_i sum_{l=i+1..j} (v_i^H v_l) T[l,j]   (i < j, same block)
__global__ void __launch_bounds__(128) bt_tprep_kernel(const c128* __restrict__ V2, const c128* __restrict__ tau2,
                                                       int kmax, int N, int gs, const int64_t* __restrict__ pass_off,
                                                       c128* __restrict__ Tneg) {
    extern __shared__ __align__(16) unsigned char tp_raw[];
    c128* Vs = reinterpret_cast<c128*>(tp_raw);  // dense window layout, Vs[r + t*96]
    c128* Gs = Vs + BT_WR * BT_P;
    c128* Ts = Gs + BT_P * (BT_P + 1);
    c128* taus = Ts + BT_P * (BT_P + 1);
    const int pass = blockIdx.y, k = blockIdx.x;
    const int j0 = pass * BT_P;
    if (j0 + 1 + k * BT_B > N - 1) return;       // no reflector of this pass reaches step k
    const int tid = threadIdx.x;
    for (int idx = tid; idx < BT_WR * BT_P; idx += 128) Vs[idx] = cmake(0.0, 0.0);
    for (int idx = tid; idx < BT_P * (BT_P + 1); idx += 128) Ts[idx] = cmake(0.0, 0.0);
    __syncthreads();
    for (int idx = tid; idx < BT_B * BT_P; idx += 128) {
        const int i = idx % BT_B, t = idx / BT_B;
        const int j = j0 + t;
        const int r0 = j + 1 + k * BT_B;
        const int len = min(BT_B, N - r0);
        if (j <= N - 2 && i < len) {
            const int64_t voff = (int64_t)j * (N - 1) - (int64_t)j * (j - 1) / 2;
            Vs[(t + i) + t * BT_WR] = V2[voff + (int64_t)k * BT_B + i];
        }
    }
    if (tid < BT_P) {
        const int j = j0 + tid;
        const int r0 = j + 1 + k * BT_B;
        taus[tid] = (j <= N - 2 && r0 <= N - 1) ? tau2[(int64_t)j * kmax + k] : cmake(0.0, 0.0);
    }
    __syncthreads();
    // Gram entries G[i][l] = v_i^H v_l for i < l inside the same GS block
    for (int idx = tid; idx < BT_P * BT_P; idx += 128) {
        const int i = idx % BT_P, l = idx / BT_P;
        c128 s = cmake(0.0, 0.0);
        if (i < l && i / gs == l / gs) {
            // overlap of rows [i, i+64) and [l, l+64): [l, i+64)
            for (int r = l; r < i + BT_B; ++r) cfmac(s, Vs[r + i * BT_WR], Vs[r + l * BT_WR]);
        }
        Gs[i + l * (BT_P + 1)] = s;
    }
    __syncthreads();
    if (tid < BT_P) {
        const int j = tid, blk0 = (j / gs) * gs;
        Ts[j + j * (BT_P + 1)] = taus[j];
        for (int i = j - 1; i >= blk0; --i) {
            c128 s = cmake(0.0, 0.0);
            for (int l = i + 1; l <= j; ++l) cfma(s, Gs[i + l * (BT_P + 1)], Ts[l + j * (BT_P + 1)]);
            const c128 ti = taus[i];
            Ts[i + j * (BT_P + 1)] = cmake(-(ti.x * s.x - ti.y * s.y), -(ti.x * s.y + ti.y * s.x));
        }
    }
    __syncthreads();
    c128* out = Tneg + (size_t)(pass_off[pass] + k) * BT_TS;
    for (int idx = tid; idx < BT_TS; idx += 128) {
        const int o = idx % BT_LDT, in = idx / BT_LDT;
        c128 v = cmake(0.0, 0.0);
        if (o < BT_P) { const c128 t = Ts[o + in * (BT_P + 1)]; v = cmake(-t.x, -t.y); }
        out[idx] = v;
    }
}

// ------------------------------------------------------------------ mbarrier / bulk-copy helpers
__device__ __forceinline__ void mbar_init(uint64_t* b, int count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(b)), "r"(count));
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint64_t* b, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(b)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t* b) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(b)) : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(uint64_t* b, uint32_t parity) {
    uint32_t ok;
    asm volatile(
        "{\n.reg .pred p;\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
        "selp.u32 %0, 1, 0, p;\n}"
        : "=r"(ok)
        : "r"(smem_u32(b)), "r"(parity)
        : "memory");
    return ok != 0;
}
__device__ __forceinline__ void mbar_wait(uint64_t* b, uint32_t parity) {
    while (!mbar_try_wait(b, parity)) {}
}
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, uint32_t bytes, uint64_t* b) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                     smem_u32(dst)),
                 "l"(src), "r"(bytes), "r"(smem_u32(b))
                 : "memory");
}
// pure (non-volatile) DMMA so that the compiler may schedule it freely
__device__ __forceinline__ void dmma_p(double (&c)[2], double a, double b) {
    asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
        : "+d"(c[0]), "+d"(c[1])
        : "d"(a), "d"(b));
}

struct BtSweepArgs {
    c128* Z; int64_t ldz;
    int N, nev;
    const c128* V2;
    const c128* Tneg;
    const int64_t* pass_off;
    int npass, nslabs;
    unsigned long long* unit_counter;   // zero on entry
    int* slab_done;                     // [nslabs], zero on entry; += 8 per finished (pass, slab)
};

// ------------------------------------------------------------------ the sweeper
// One (pass, k) step on the register window.  GS = reflectors per compact-WY block (8, 16 or 32).
template <int GS>
__device__ __forceinline__ void bt_apply_step(const c128* __restrict__ Vs, const c128* __restrict__ Ts,
                                              double (&zr)[BT_NBLK][2], double (&zi)[BT_NBLK][2], int g, int t,
                                              bool tail, int nrows) {
    constexpr int NB = GS / 8;          // column blocks per WY block
    constexpr int NSUB = BT_P / GS;
#pragma unroll
    for (int s = NSUB - 1; s >= 0; --s) {
        const int cb0 = s * NB;
        // ---- Y1 = V^H Z   (m = column of Z, n = reflector, k = row)
        double y1r[NB][2][2], y1i[NB][2][2];   // [col block][k-step parity h][frag]
#pragma unroll
        for (int c = 0; c < NB; ++c)
#pragma unroll
            for (int h = 0; h < 2; ++h) y1r[c][h][0] = y1r[c][h][1] = y1i[c][h][0] = y1i[c][h][1] = 0.0;
#pragma unroll
        for (int p = cb0; p < cb0 + NB + 8; ++p) {
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                const double ar = zr[p][h], ai = zi[p][h], nar = -ar;
#pragma unroll
                for (int c = 0; c < NB; ++c) {
                    const int cb = cb0 + c;
                    if (p >= cb && p <= cb + 8) {
                        const c128 v = Vs[(8 * p + 2 * t + h) + (8 * cb + g) * BT_LDV];
                        // (ar + i ai) * (v.x - i v.y)
                        dmma_p(y1r[c][h], ar, v.x);
                        dmma_p(y1i[c][h], ai, v.x);
                        dmma_p(y1r[c][h], ai, v.y);
                        dmma_p(y1i[c][h], nar, v.y);
                    }
                }
            }
        }
        double ar1[NB][2], ai1[NB][2];      // Y1 as the A operand of the T product: element h = reflector 8c+2t+h
#pragma unroll
        for (int c = 0; c < NB; ++c)
#pragma unroll
            for (int e = 0; e < 2; ++e) {
                ar1[c][e] = y1r[c][0][e] + y1r[c][1][e];
                ai1[c][e] = y1i[c][0][e] + y1i[c][1][e];
            }
        // ---- Y = (-T) Y1   (m = column of Z, n = output reflector, k = input reflector >= output)
        double yr[NB][2], yi[NB][2];
#pragma unroll
        for (int co = 0; co < NB; ++co) {
            yr[co][0] = yr[co][1] = yi[co][0] = yi[co][1] = 0.0;
#pragma unroll
            for (int ci = co; ci < NB; ++ci)
#pragma unroll
                for (int h = 0; h < 2; ++h) {
                    const c128 tt = Ts[(8 * (cb0 + co) + g) + (8 * (cb0 + ci) + 2 * t + h) * BT_LDT];
                    const double ar = ar1[ci][h], ai = ai1[ci][h], nai = -ai;
                    dmma_p(yr[co], ar, tt.x);
                    dmma_p(yi[co], ai, tt.x);
                    dmma_p(yr[co], nai, tt.y);
                    dmma_p(yi[co], ar, tt.y);
                }
        }
        // ---- Z += Y V   (m = column of Z, n = row, k = reflector)
#pragma unroll
        for (int c = 0; c < NB; ++c) {
            const int cb = cb0 + c;
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                const double ar = yr[c][h], ai = yi[c][h], nai = -ai;
#pragma unroll
                for (int p = cb; p <= cb + 8; ++p) {
                    const c128 v = Vs[(8 * p + g) + (8 * cb + 2 * t + h) * BT_LDV];
                    dmma_p(zr[p], ar, v.x);
                    dmma_p(zi[p], ai, v.x);
                    dmma_p(zr[p], nai, v.y);
                    dmma_p(zi[p], ar, v.y);
                }
            }
        }
        if (tail) {
            // rows beyond the matrix are virtual: keep them zero (stale V rows may have touched them)
#pragma unroll
            for (int p = cb0; p < cb0 + NB + 8; ++p)
#pragma unroll
                for (int e = 0; e < 2; ++e)
                    if (8 * p + 2 * t + e >= nrows) { zr[p][e] = 0.0; zi[p][e] = 0.0; }
        }
    }
}

template <int GS>
__global__ void __launch_bounds__(BT_NT, 1) bt_sweep_kernel(const BtSweepArgs a) {
    extern __shared__ __align__(128) unsigned char bt_raw[];
    c128* Vring = reinterpret_cast<c128*>(bt_raw);
    c128* Tring = Vring + (size_t)BT_STAGES * BT_VS;
    BtHeader* hdr = reinterpret_cast<BtHeader*>(Tring + (size_t)BT_STAGES * BT_TS);
    uint64_t* full = reinterpret_cast<uint64_t*>(hdr + BT_STAGES);
    uint64_t* empty = full + BT_STAGES;

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    for (int idx = tid; idx < BT_STAGES * (BT_VS + BT_TS); idx += BT_NT) Vring[idx] = cmake(0.0, 0.0);
    if (tid == 0) {
        for (int s = 0; s < BT_STAGES; ++s) { mbar_init(&full[s], 1); mbar_init(&empty[s], BT_CWARPS); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    __syncthreads();

    const int N = a.N;
    if (warp == BT_CWARPS) {
        // =============================== producer warp (one lane)
        if (lane != 0) return;
        uint32_t it = 0;
        const unsigned long long total = (unsigned long long)a.npass * a.nslabs;
        for (;;) {
            const unsigned long long u = atomicAdd(a.unit_counter, 1ULL);
            if (u >= total) {
                const int slot = it % BT_STAGES;
                mbar_wait(&empty[slot], ((it / BT_STAGES) & 1) ^ 1);
                hdr[slot].flags = 4;
                mbar_arrive(&full[slot]);
                break;
            }
            const int round = (int)(u / a.nslabs);
            const int pass = a.npass - 1 - round;
            const int slab = (int)(u % a.nslabs);
            const int j0 = pass * BT_P;
            // all eight warps of the unit (pass+1, slab) must have stored their rows
            while (*(volatile int*)(a.slab_done + slab) < BT_CWARPS * round) {}
            __threadfence();
            const int nk = (N - 1 - j0 + BT_B - 1) / BT_B;
            const c128* Tn = a.Tneg + (size_t)a.pass_off[pass] * BT_TS;
            for (int k = 0; k < nk; ++k, ++it) {
                const int slot = it % BT_STAGES;
                mbar_wait(&empty[slot], ((it / BT_STAGES) & 1) ^ 1);
                BtHeader hh;
                hh.j0 = j0; hh.k = k; hh.slab = slab;
                hh.flags = (k == 0 ? 1 : 0) | (k == nk - 1 ? 2 : 0);
                hdr[slot] = hh;
                uint32_t bytes = BT_TS * sizeof(c128);
                c128* Vs = Vring + (size_t)slot * BT_VS;
#pragma unroll 1
                for (int t = 0; t < BT_P; ++t) {
                    const int j = j0 + t;
                    const int len = min(BT_B, N - (j + 1 + k * BT_B));
                    if (j <= N - 2 && len > 0) bytes += len * (int)sizeof(c128);
                }
                mbar_arrive_expect_tx(&full[slot], bytes);
#pragma unroll 1
                for (int t = 0; t < BT_P; ++t) {
                    const int j = j0 + t;
                    const int len = min(BT_B, N - (j + 1 + k * BT_B));
                    if (j <= N - 2 && len > 0) {
                        const int64_t voff = (int64_t)j * (N - 1) - (int64_t)j * (j - 1) / 2;
                        bulk_g2s(Vs + t * (BT_LDV + 1), a.V2 + voff + (int64_t)k * BT_B, len * (int)sizeof(c128), &full[slot]);
                    }
                }
                bulk_g2s(Tring + (size_t)slot * BT_TS, Tn + (size_t)k * BT_TS, BT_TS * sizeof(c128), &full[slot]);
            }
        }
        return;
    }

    // =================================== consumer warps
    const int g = lane >> 2, t = lane & 3;
    double zr[BT_NBLK][2], zi[BT_NBLK][2];
#pragma unroll
    for (int p = 0; p < BT_NBLK; ++p) zr[p][0] = zr[p][1] = zi[p][0] = zi[p][1] = 0.0;

    for (uint32_t it = 0;; ++it) {
        const int slot = it % BT_STAGES;
        mbar_wait(&full[slot], (it / BT_STAGES) & 1);
        const BtHeader hh = hdr[slot];
        if (hh.flags & 4) break;
        const int R0 = hh.j0 + 1 + hh.k * BT_B;
        const int col = hh.slab * BT_SLAB + warp * 8 + g;
        const bool colok = col < a.nev;
        c128* Zc = a.Z + (int64_t)col * a.ldz;
        const int nrows = N - R0;                 // valid rows of the window (>= 1)
        if (hh.flags & 1) {
#pragma unroll
            for (int p = 0; p < BT_NBLK; ++p)
#pragma unroll
                for (int e = 0; e < 2; ++e) {
                    const int w = 8 * p + 2 * t + e;
                    c128 v = cmake(0.0, 0.0);
                    if (colok && w < nrows) v = __ldcg(Zc + R0 + w);
                    zr[p][e] = v.x; zi[p][e] = v.y;
                }
        }
        const c128* Vs = Vring + (size_t)slot * BT_VS;
        const c128* Ts = Tring + (size_t)slot * BT_TS;
        bt_apply_step<GS>(Vs, Ts, zr, zi, g, t, nrows < BT_WR, nrows);
        __syncwarp();
        if (lane == 0) mbar_arrive(&empty[slot]);
        if (hh.flags & 2) {
            // last step of the unit: store the whole window
#pragma unroll
            for (int p = 0; p < BT_NBLK; ++p)
#pragma unroll
                for (int e = 0; e < 2; ++e) {
                    const int w = 8 * p + 2 * t + e;
                    if (colok && w < nrows) Zc[R0 + w] = cmake(zr[p][e], zi[p][e]);
                }
            __threadfence();
            __syncwarp();
            if (lane == 0) atomicAdd(a.slab_done + hh.slab, 1);
        } else {
            // store the finished top 64 rows, slide the window, fetch the next 64 rows
#pragma unroll
            for (int p = 0; p < 8; ++p)
#pragma unroll
                for (int e = 0; e < 2; ++e) {
                    const int w = 8 * p + 2 * t + e;
                    if (colok && w < nrows) Zc[R0 + w] = cmake(zr[p][e], zi[p][e]);
                }
#pragma unroll
            for (int p = 0; p < BT_NBLK - 8; ++p)
#pragma unroll
                for (int e = 0; e < 2; ++e) { zr[p][e] = zr[p + 8][e]; zi[p][e] = zi[p + 8][e]; }
#pragma unroll
            for (int p = BT_NBLK - 8; p < BT_NBLK; ++p)
#pragma unroll
                for (int e = 0; e < 2; ++e) {
                    const int w = 8 * p + 2 * t + e + BT_B;       // row offset from the old R0
                    c128 v = cmake(0.0, 0.0);
                    if (colok && w < nrows) v = __ldcg(Zc + R0 + w);
                    zr[p][e] = v.x; zi[p][e] = v.y;
                }
        }
    }
}

template <int GS>
static int bt_launch_sweep(eigh_handle_s* h, const BtSweepArgs& a, cudaStream_t s) {
    auto kern = bt_sweep_kernel<GS>;
    static bool attr = false;
    if (!attr) {
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)BT_SMEM);
        if (e != cudaSuccess) return 1000 + (int)e;
        attr = true;
    }
    int grid = h->num_sms;
    const long long units = (long long)a.npass * a.nslabs;
    if (grid > units) grid = (int)units;
    kern<<<grid, BT_NT, BT_SMEM, s>>>(a);
    ++h->launches;
    const cudaError_t e = cudaGetLastError();
    return e != cudaSuccess ? 1000 + (int)e : 0;
}

int phase_backtransform_band(eigh_handle_s* h, const double* Qt, int64_t ldq, c128* Z, int64_t ldz, cudaStream_t s) {
    const int N = (int)h->N, nev = (int)h->nev;
    if (h->b != BT_B) return set_err(h, -100, "band back-transformation is built for band width %d", BT_B);
    const WsPlan& pl = h->plan;
    const double* sgn = ws_ptr<double>(h, pl.sgn);
    bt_expand_kernel<<<dim3((unsigned)ceil_div(N, 256), (unsigned)nev), 256, 0, s>>>(Qt, ldq, sgn, N, nev, Z, ldz);
    ++h->launches;
    if (N < 2) return 0;
    const int npass = (int)bt_npass(N);
    const int nslabs = (int)ceil_div(nev, BT_SLAB);
    char* scr = ws_ptr<char>(h, pl.bt) + round_up((size_t)h->b * nev * sizeof(c128), 256);
    int64_t* pass_off = reinterpret_cast<int64_t*>(scr);
    unsigned long long* counter = reinterpret_cast<unsigned long long*>(pass_off + npass + 4);
    int* slab_done = reinterpret_cast<int*>(counter + 2);
    c128* Tneg = ws_ptr<c128>(h, pl.btT);
    EIGH_CUDA_OK(cudaMemsetAsync(counter, 0, 16 + (size_t)(nslabs + 8) * sizeof(int), s));
    bt_pass_off_kernel<<<1, 32, 0, s>>>(N, npass, pass_off);
    const int kmax = (int)bc_kmax(h);
    int gs = h->g;
    if (gs != 8 && gs != 16 && gs != 32) gs = 8;
    const size_t tp_smem = (size_t)(BT_WR * BT_P + 2 * BT_P * (BT_P + 1) + BT_P) * sizeof(c128);
    static bool tp_attr = false;
    if (!tp_attr) {
        EIGH_CUDA_OK(cudaFuncSetAttribute(bt_tprep_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)tp_smem));
        tp_attr = true;
    }
    bt_tprep_kernel<<<dim3((unsigned)kmax, (unsigned)npass), 128, tp_smem, s>>>(ws_ptr<c128>(h, pl.V2), ws_ptr<c128>(h, pl.tau2),
                                                                           kmax, N, gs, pass_off, Tneg);
    h->launches += 2;
    BtSweepArgs a;
    a.Z = Z; a.ldz = ldz; a.N = N; a.nev = nev; a.V2 = ws_ptr<c128>(h, pl.V2); a.Tneg = Tneg; a.pass_off = pass_off;
    a.npass = npass; a.nslabs = nslabs; a.unit_counter = counter; a.slab_done = slab_done;
    int rc;
    if (gs == 8) rc = bt_launch_sweep<8>(h, a, s);
    else if (gs == 16) rc = bt_launch_sweep<16>(h, a, s);
    else rc = bt_launch_sweep<32>(h, a, s);
    return rc;
}

}  // namespace eigh
