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
//    1-D bulk async copies (cp.async.bulk, SASS UBLKCP) into a 3-stage ring guarded by full/empty
//    mbarriers.  There is no producer warp (a ninth warp would cap every thread at 168 registers:
//    three warps on one SM sub-partition): lane 0 of warp 0 issues the copies of stage it+2 at the
//    top of step it.  The 8 warps never meet at a CTA barrier.
//    Shared-memory leading dimensions are odd (97, 33), which makes both fragment access patterns
//    (row-fastest for V^H Z, column-fastest for V Y) conflict-free for 128-bit loads.
//  * Z rows enter and leave the register window straight from/to global memory: the window slides
//    down by 64 rows per step, so every row of Z is read once and written once per pass.  The 64
//    rows of the next step are fetched into a second register set BEFORE the products of the
//    current step, so their latency is hidden behind ~30k cycles of DMMA work.
//  * Units are handed out by an atomic counter.  Dependencies are per (pass, slab, warp) -- a warp
//    owns its 8 columns for the whole unit, so it only ever depends on the same warp index of the
//    unit (pass+1, slab): step k of pass p-1 reads rows that pass p finalises in its step k.  Every
//    warp publishes "steps completed" with a release store (delayed by one step so that the fence
//    finds the stores already drained) and polls its predecessor with ld.acquire.
//  * Unit order: groups of `chain` consecutive passes; inside a group slab-major, so that the
//    chain members of one slab run concurrently on neighbouring CTAs, a few steps apart, and the
//    followers read from L2 what the leader has just written (HBM traffic / chain).
#include "eigh_internal.h"

namespace eigh {

constexpr bool BT_QPLANE = true;    // stage tiles carry q = vx - vy (a third bulk copy, 16 KB): no V-side adds in the two 3-product forms
constexpr bool BT_Y1_SPLIT = false;  // Y1 = V^H Z: one accumulator chain per 3M sum (false) or one per k-step parity (true: 6 more adds per block)
constexpr int BT_RING8 = 3;         // stages of the ring for GS = 8 (with the q plane there is room for three)
constexpr int BT_B = 64;            // band width (reflector length)
constexpr int BT_P = 32;            // sweeps per pass
constexpr int BT_WR = BT_B + BT_P;  // window rows (96)
constexpr int BT_NBLK = BT_WR / 8;  // 12 row blocks
constexpr int BT_LDV = BT_B - 1;    // 63: element (window row R, reflector c) of a stage at 63 c + R (valid for 0 <= R - c < 64),
                                    // i.e. the stage is the plain [32][64] tile of the reflector storage; odd => conflict-free
constexpr int BT_LDT = BT_P + 1;    // 33, odd
constexpr int BT_VS = BT_B * BT_P;          // c128 per V stage (32 KB)
constexpr int BT_TS = BT_LDT * BT_P;        // c128 per T stage
constexpr int BT_LDZ = BT_B + 1;            // 65, odd: per-warp staging of the 64 incoming rows of 8 columns
constexpr int BT_ZS = 8 * BT_LDZ;           // c128 per warp
// compact -T of one (pass, k) step for WY blocks of GS reflectors: 32/GS blocks [GS x GS], ld GS+1
__host__ __device__ constexpr int bt_tsz(int gs) { return BT_P * (gs + 1); }
__host__ __device__ constexpr bool bt_qplane(int gs) { return BT_QPLANE && gs == 8; }   // 16 / 32: no shared memory left for it
__host__ __device__ constexpr int bt_stages(int gs) { return gs == 8 ? BT_RING8 : 3; }
constexpr int BT_CWARPS = 8;                // warps per CTA (all of them consumers)
constexpr int BT_NT = 32 * BT_CWARPS;
constexpr int BT_SLAB = 8 * BT_CWARPS;      // 64 columns per unit

struct BtHeader { int j0, k, slab, flags, pass, nk_pred, pad0, pad1; };   // flags: 1 first step of unit, 2 last step, 4 terminate
__host__ __device__ constexpr size_t bt_smem(int gs) {
    return (size_t)bt_stages(gs) * (BT_VS + bt_tsz(gs)) * sizeof(c128) + (size_t)BT_CWARPS * BT_ZS * sizeof(c128) +
           (bt_qplane(gs) ? (size_t)bt_stages(gs) * BT_VS * sizeof(double) : 0) +
           bt_stages(gs) * sizeof(BtHeader) + (2 * bt_stages(gs) + BT_CWARPS) * sizeof(uint64_t) + 64;
}

static inline int64_t bt_npass(int64_t N) { return v2_npass(N); }

size_t bt_tneg_bytes(int64_t N) {
    // stages = sum over passes of ceil((N-1-j0)/64)  <=  npass * kmax
    int64_t st = 0;
    for (int64_t p = 0; p < bt_npass(N); ++p) st += ceil_div(N - 1 - p * BT_P, BT_B);
    return (size_t)st * BT_TS * sizeof(c128) + 256;
}
size_t bt_scratch_bytes(const eigh_handle_s* h) {
    // S4b's Y + pass offsets + unit counter + per (pass, slab, warp) progress counters
    const size_t y = (size_t)h->b * h->nev * sizeof(c128);
    const size_t prog = (size_t)bt_npass(h->N) * ceil_div(h->nev, BT_SLAB) * BT_CWARPS * sizeof(int);
    return y + (size_t)(bt_npass(h->N) + 8) * sizeof(int64_t) + prog + 8192;
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
            Vs[(t + i) + t * BT_WR] = V2[((pass_off[pass] + k) * BT_P + t) * BT_B + i];
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
    // compact layout: block s = reflectors [s gs, (s+1) gs); element (o, in) of block s at s gs (gs+1) + o + in (gs+1)
    const int ldc = gs + 1;
    for (int idx = tid; idx < BT_P * ldc; idx += 128) {
        const int blk = idx / (gs * ldc), rem = idx % (gs * ldc);
        const int o = rem % ldc, in = rem / ldc;
        c128 v = cmake(0.0, 0.0);
        if (o < gs) { const c128 t = Ts[(blk * gs + o) + (blk * gs + in) * (BT_P + 1)]; v = cmake(-t.x, -t.y); }
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
__device__ __forceinline__ void bulk_s2g(void* gdst, const void* ssrc, uint32_t bytes) {
    asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(gdst), "r"(smem_u32(ssrc)), "r"(bytes)
                 : "memory");
}
__device__ __forceinline__ void bulk_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void bulk_wait_read() { asm volatile("cp.async.bulk.wait_group.read %0;" ::"n"(N) : "memory"); }
template <int N>
__device__ __forceinline__ void bulk_wait() { asm volatile("cp.async.bulk.wait_group %0;" ::"n"(N) : "memory"); }
// pure (non-volatile) DMMA so that the compiler may schedule it freely
__device__ __forceinline__ void dmma_p(double (&c)[2], double a, double b) {
    asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
        : "+d"(c[0]), "+d"(c[1])
        : "d"(a), "d"(b));
}

// q = Re v - Im v for every stored reflector element (the third operand of the 3-product forms, formed once here instead
// of once per warp and use inside the sweep)
__global__ void bt_vq_kernel(const c128* __restrict__ V2, double* __restrict__ q, int64_t n) {
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
        const c128 v = V2[i];
        q[i] = v.x - v.y;
    }
}
size_t bt_vq_bytes(int64_t N) { return BT_QPLANE ? (size_t)(v2_total_stages(N) * BT_VS + 64) * sizeof(double) : 0; }

struct BtSweepArgs {
    c128* Z; int64_t ldz;
    int N, nev;
    const c128* V2;
    const double* V2q;                  // q = Re v - Im v of every element of V2 (same tile-major layout)
    const c128* Tneg;
    const int64_t* pass_off;
    int npass, nslabs, chain;
    unsigned long long* unit_counter;   // zero on entry
    int* prog;                          // [npass][nslabs][8], zero on entry: steps completed by (pass, slab, warp)
};

__device__ __forceinline__ int bt_ld_acquire(const int* p) {
    int v;
    asm volatile("ld.acquire.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void bt_st_release(int* p, int v) {
    asm volatile("st.release.gpu.global.s32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}

// ------------------------------------------------------------------ the sweeper
// One (pass, k) step on the register window.  GS = reflectors per compact-WY block (8, 16 or 32).
template <int GS, int S_HI, int S_LO>
__device__ __forceinline__ void bt_apply_step(const c128* __restrict__ Vs, const double* __restrict__ Qs,
                                              const c128* __restrict__ Ts,
                                              double (&zr)[BT_NBLK][2], double (&zi)[BT_NBLK][2], int g, int t,
                                              bool tail, int nrows) {
    constexpr int NB = GS / 8;          // column blocks per WY block
    constexpr int NSUB = BT_P / GS;
#pragma unroll
    static_assert(S_HI < NSUB && S_LO >= 0, "sub-block range");
#pragma unroll
    for (int s = S_HI; s >= S_LO; --s) {
        const int cb0 = s * NB;
        // ---- Y1 = V^H Z   (m = column of Z, n = reflector, k = row)
        // 3M form of the complex product (three real DMMAs per complex multiply-add instead of four; the sums
        // run over all 72 rows before they are combined):  with z = ar + i ai and conj(v) = v.x - i v.y,
        //   S1 = sum ar v.x,  S2 = sum ai v.y,  S3 = sum (ar + ai)(v.x - v.y);   Re = S1 + S2,  Im = S3 - S1 + S2.
        double s1[NB][2][2], s2[NB][2][2], s3[NB][2][2];   // [col block][k-step parity h][frag]
#pragma unroll
        for (int c = 0; c < NB; ++c)
#pragma unroll
            for (int h = 0; h < 2; ++h)
                s1[c][h][0] = s1[c][h][1] = s2[c][h][0] = s2[c][h][1] = s3[c][h][0] = s3[c][h][1] = 0.0;
#pragma unroll
        for (int p = cb0; p < cb0 + NB + 8; ++p) {
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                const double ar = zr[p][h], ai = zi[p][h], as = ar + ai;
#pragma unroll
                for (int c = 0; c < NB; ++c) {
                    const int cb = cb0 + c;
                    if (p >= cb && p <= cb + 8) {
                        // window row R = 8p+2t+h, reflector c = 8cb+g: inside the parallelogram iff 0 <= R - c < 64
                        c128 v = cmake(0.0, 0.0);
                        double qv = 0.0;
                        if ((p != cb || 2 * t + h >= g) && (p != cb + 8 || 2 * t + h < g)) {
                            v = Vs[(8 * p + 2 * t + h) + (8 * cb + g) * BT_LDV];
                            if constexpr (bt_qplane(GS)) qv = Qs[(8 * p + 2 * t + h) + (8 * cb + g) * BT_LDV];
                        }
                        if constexpr (!bt_qplane(GS)) qv = v.x - v.y;
                        dmma_p(s1[c][BT_Y1_SPLIT ? h : 0], ar, v.x);
                        dmma_p(s2[c][BT_Y1_SPLIT ? h : 0], ai, v.y);
                        dmma_p(s3[c][BT_Y1_SPLIT ? h : 0], as, qv);
                    }
                }
            }
        }
        double ar1[NB][2], ai1[NB][2];      // Y1 as the A operand of the T product: element h = reflector 8c+2t+h
#pragma unroll
        for (int c = 0; c < NB; ++c)
#pragma unroll
            for (int e = 0; e < 2; ++e) {
                const double t1 = BT_Y1_SPLIT ? s1[c][0][e] + s1[c][1][e] : s1[c][0][e];
                const double t2 = BT_Y1_SPLIT ? s2[c][0][e] + s2[c][1][e] : s2[c][0][e];
                const double t3 = BT_Y1_SPLIT ? s3[c][0][e] + s3[c][1][e] : s3[c][0][e];
                ar1[c][e] = t1 + t2;
                ai1[c][e] = (t3 - t1) + t2;
            }
        // ---- Y = (-T) Y1   (m = column of Z, n = output reflector, k = input reflector >= output)
        double yr[NB][2], yi[NB][2];
#pragma unroll
        for (int co = 0; co < NB; ++co) {
            // two accumulator pairs (one per k-step parity h): the dependent chain Y1 -> Y -> Z is two DMMAs deep instead of four
            double yra[2] = {0.0, 0.0}, yia[2] = {0.0, 0.0}, yrb[2] = {0.0, 0.0}, yib[2] = {0.0, 0.0};
#pragma unroll
            for (int ci = co; ci < NB; ++ci)
#pragma unroll
                for (int h = 0; h < 2; ++h) {
                    const c128 tt = Ts[s * GS * (GS + 1) + (8 * co + g) + (8 * ci + 2 * t + h) * (GS + 1)];
                    const double ar = ar1[ci][h], ai = ai1[ci][h], nai = -ai;
                    if (h == 0) {
                        dmma_p(yra, ar, tt.x);
                        dmma_p(yia, ai, tt.x);
                        dmma_p(yra, nai, tt.y);
                        dmma_p(yia, ar, tt.y);
                    } else {
                        dmma_p(yrb, ar, tt.x);
                        dmma_p(yib, ai, tt.x);
                        dmma_p(yrb, nai, tt.y);
                        dmma_p(yib, ar, tt.y);
                    }
                }
            yr[co][0] = yra[0] + yrb[0]; yr[co][1] = yra[1] + yrb[1];
            yi[co][0] = yia[0] + yib[0]; yi[co][1] = yia[1] + yib[1];
        }
        // ---- Z += Y V   (m = column of Z, n = row, k = reflector)
        if constexpr (bt_qplane(GS)) {
        // Three real products per complex multiply-add with the precomputed q = vx - vy:  with y = ar + i ai,
        //   k1 = ai q,  k2 = (ar - ai) vx,  k3 = (ar + ai) vy;   Re(y v) = k2 + k1,  Im(y v) = k3 + k1.
#pragma unroll
        for (int c = 0; c < NB; ++c) {
            const int cb = cb0 + c;
            double ai[2], dm[2], sp[2];
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                ai[h] = yi[c][h];
                dm[h] = yr[c][h] - yi[c][h];
                sp[h] = yr[c][h] + yi[c][h];
            }
#pragma unroll
            for (int p = cb; p <= cb + 8; ++p) {
                double k1[2] = {0.0, 0.0};
#pragma unroll
                for (int h = 0; h < 2; ++h) {
                    c128 v = cmake(0.0, 0.0);
                    double qv = 0.0;
                    if ((p != cb || g >= 2 * t + h) && (p != cb + 8 || g < 2 * t + h)) {
                        v = Vs[(8 * p + g) + (8 * cb + 2 * t + h) * BT_LDV];
                        qv = Qs[(8 * p + g) + (8 * cb + 2 * t + h) * BT_LDV];
                    }
                    dmma_p(k1, ai[h], qv);
                    dmma_p(zr[p], dm[h], v.x);
                    dmma_p(zi[p], sp[h], v.y);
                }
                zr[p][0] += k1[0]; zr[p][1] += k1[1];
                zi[p][0] += k1[0]; zi[p][1] += k1[1];
            }
        }
        } else {
        // Three real products per complex multiply-add (Gauss): with y = ar + i ai and v = vx + i vy,
        //   k1 = ar (vx + vy),  k2 = (ai - ar) vx,  k3 = (ar + ai) vy;   Re(y v) = k1 - k3,  Im(y v) = k1 + k2.
        // k2 and k3 accumulate straight into zi and zr; k1 is summed over the block's 8 reflectors and added to both.
#pragma unroll
        for (int c = 0; c < NB; ++c) {
            const int cb = cb0 + c;
            double ar[2], df[2], ns[2];
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                ar[h] = yr[c][h];
                df[h] = yi[c][h] - yr[c][h];
                ns[h] = -(yr[c][h] + yi[c][h]);
            }
#pragma unroll
            for (int p = cb; p <= cb + 8; ++p) {
                double k1[2] = {0.0, 0.0};
#pragma unroll
                for (int h = 0; h < 2; ++h) {
                    c128 v = cmake(0.0, 0.0);
                    if ((p != cb || g >= 2 * t + h) && (p != cb + 8 || g < 2 * t + h))
                        v = Vs[(8 * p + g) + (8 * cb + 2 * t + h) * BT_LDV];
                    dmma_p(k1, ar[h], v.x + v.y);
                    dmma_p(zi[p], df[h], v.x);
                    dmma_p(zr[p], ns[h], v.y);
                }
                zr[p][0] += k1[0]; zr[p][1] += k1[1];
                zi[p][0] += k1[0]; zi[p][1] += k1[1];
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

// Stage producer state (uniform over warp 0; only lane 0 touches shared/global memory).
struct BtProducer {
    uint32_t it;       // stages produced so far
    int pass, slab, k, nk;
    bool done;
};

template <int GS>
__global__ void __launch_bounds__(BT_NT, 1) bt_sweep_kernel(const BtSweepArgs a) {
    extern __shared__ __align__(128) unsigned char bt_raw[];
    c128* Vring = reinterpret_cast<c128*>(bt_raw);
    constexpr int BT_STAGES = bt_stages(GS), BT_TSZ = bt_tsz(GS);
    c128* Tring = Vring + (size_t)BT_STAGES * BT_VS;
    c128* Zstage = Tring + (size_t)BT_STAGES * BT_TSZ;
    double* Qring = reinterpret_cast<double*>(Zstage + (size_t)BT_CWARPS * BT_ZS);
    BtHeader* hdr = reinterpret_cast<BtHeader*>(Qring + (bt_qplane(GS) ? (size_t)BT_STAGES * BT_VS : 0));
    uint64_t* full = reinterpret_cast<uint64_t*>(hdr + BT_STAGES);
    uint64_t* empty = full + BT_STAGES;
    uint64_t* zfull = empty + BT_STAGES;          // one per warp

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    for (int idx = tid; idx < BT_STAGES * (BT_VS + BT_TSZ) + BT_CWARPS * BT_ZS; idx += BT_NT) Vring[idx] = cmake(0.0, 0.0);
    if (bt_qplane(GS))
        for (int idx = tid; idx < BT_STAGES * BT_VS; idx += BT_NT) Qring[idx] = 0.0;
    if (tid == 0) {
        for (int s = 0; s < BT_STAGES; ++s) { mbar_init(&full[s], 1); mbar_init(&empty[s], BT_CWARPS); }
        for (int w = 0; w < BT_CWARPS; ++w) mbar_init(&zfull[w], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    __syncthreads();

    const int N = a.N;
    const unsigned long long units_per_group = (unsigned long long)a.nslabs * a.chain;
    const unsigned long long ngroups = (unsigned long long)((a.npass + a.chain - 1) / a.chain);
    const unsigned long long total = ngroups * units_per_group;

    BtProducer pr;
    pr.it = 0; pr.pass = 0; pr.slab = 0; pr.k = 0; pr.nk = 0; pr.done = false;

    // produce one stage (warp 0 only; all lanes keep the state, lane 0 acts)
    auto produce = [&]() {
        if (pr.done) return;
        while (pr.k == pr.nk) {
            unsigned long long u = 0;
            if (lane == 0) u = atomicAdd(a.unit_counter, 1ULL);
            u = __shfl_sync(0xffffffffu, u, 0);
            if (u >= total) {
                const int slot = pr.it % BT_STAGES;
                if (lane == 0) {
                    mbar_wait(&empty[slot], ((pr.it / BT_STAGES) & 1) ^ 1);
                    hdr[slot].flags = 4;
                    mbar_arrive(&full[slot]);
                }
                ++pr.it;
                pr.done = true;
                return;
            }
            const unsigned long long g = u / units_per_group, rem = u % units_per_group;
            pr.slab = (int)(rem / a.chain);
            pr.pass = a.npass - 1 - (int)(g * a.chain + rem % a.chain);
            pr.k = 0;
            pr.nk = (pr.pass >= 0) ? (N - 1 - pr.pass * BT_P + BT_B - 1) / BT_B : 0;   // padding units of the last group are empty
        }
        const int slot = pr.it % BT_STAGES;
        {
            const int j0 = pr.pass * BT_P, k = pr.k;
            if (lane == 0) {
                mbar_wait(&empty[slot], ((pr.it / BT_STAGES) & 1) ^ 1);
                BtHeader hh;
                hh.j0 = j0; hh.k = k; hh.slab = pr.slab; hh.pass = pr.pass;
                hh.flags = (k == 0 ? 1 : 0) | (k == pr.nk - 1 ? 2 : 0);
                hh.nk_pred = (pr.pass + 1 < a.npass) ? (N - 1 - (pr.pass + 1) * BT_P + BT_B - 1) / BT_B : 0;
                hh.pad0 = hh.pad1 = 0;
                hdr[slot] = hh;
                mbar_arrive_expect_tx(&full[slot], (uint32_t)((BT_VS + BT_TSZ) * sizeof(c128) + (bt_qplane(GS) ? BT_VS * sizeof(double) : 0)));
                // the 32 reflectors of (pass, k) are one contiguous, zero-padded 32 KB tile; -T is 32 (GS+1) elements
                const int64_t stage = a.pass_off[pr.pass] + k;
                bulk_g2s(Vring + (size_t)slot * BT_VS, a.V2 + stage * BT_VS, BT_VS * sizeof(c128), &full[slot]);
                bulk_g2s(Tring + (size_t)slot * BT_TSZ, a.Tneg + stage * BT_TS, BT_TSZ * sizeof(c128), &full[slot]);
                if (bt_qplane(GS))
                    bulk_g2s(Qring + (size_t)slot * BT_VS, a.V2q + stage * BT_VS, BT_VS * sizeof(double), &full[slot]);
            }
        }
        ++pr.it;
        ++pr.k;
    };

    if (warp == 0)
        for (int s = 0; s < BT_STAGES - 1; ++s) produce();

    const int g = lane >> 2, t = lane & 3;
    double zr[BT_NBLK][2], zi[BT_NBLK][2];
#pragma unroll
    for (int p = 0; p < BT_NBLK; ++p) zr[p][0] = zr[p][1] = zi[p][0] = zi[p][1] = 0.0;
    uint32_t zphase = 0;
    int pred_seen = 0;                  // progress of the predecessor unit as last observed by this warp

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
        const bool last = (hh.flags & 2) != 0;
        int* myprog = a.prog + ((size_t)hh.pass * a.nslabs + hh.slab) * BT_CWARPS + warp;
        const int* predprog = myprog + (size_t)a.nslabs * BT_CWARPS;     // same warp of unit (pass+1, slab)
        c128* Zs = Zstage + (size_t)warp * BT_ZS;
        const int mycol = hh.slab * BT_SLAB + warp * 8 + lane;           // column served by lanes 0..7 in bulk copies
        const bool issuer = lane < 8 && mycol < a.nev;
        if (hh.flags & 1) {
            // first step of the unit: the whole 96-row window straight from global memory.  Its last rows are
            // finalised by step 0 of the predecessor.
            pred_seen = 0;
            if (hh.nk_pred > 0) {
                int v = 0;
                if (lane == 0) do { v = bt_ld_acquire(predprog); } while (v < 1);
                pred_seen = __shfl_sync(0xffffffffu, v, 0);
                asm volatile("fence.proxy.async.global;" ::: "memory");  // rows were written through the async proxy
            }
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
        const double* Qs = Qring + (bt_qplane(GS) ? (size_t)slot * BT_VS : 0);
        const c128* Ts = Tring + (size_t)slot * BT_TSZ;
        constexpr int NSUB = BT_P / GS;
        bt_apply_step<GS, NSUB - 1, NSUB - 1>(Vs, Qs, Ts, zr, zi, g, t, nrows < BT_WR, nrows);
        // ---- prefetch the 64 rows that enter the window after this step: one 1-D bulk copy per column into
        //      this warp's staging tile (no registers, no LSU queue entries held across the step).  They are
        //      finalised by step k+1 of the predecessor.
        const int nin = last ? 0 : min(BT_B, nrows - BT_WR);          // incoming rows (may be <= 0 near the end)
        if (nin > 0) {
            if (hh.nk_pred > 0) {
                // the predecessor publishes every eighth step: one acquire usually covers the next steps too, so the
                // counter is only read again when the value seen last is not enough
                const int need = min(hh.k + 2, hh.nk_pred);
                if (pred_seen < need) {
                    int v = 0;
                    if (lane == 0) do { v = bt_ld_acquire(predprog); } while (v < need);
                    pred_seen = __shfl_sync(0xffffffffu, v, 0);
                }
            }
            if (lane < 8) bulk_wait_read<0>();                         // the tile's previous bulk stores have read it
            if (lane == 0) {
                int ncol = min(8, a.nev - (hh.slab * BT_SLAB + warp * 8));
                if (ncol < 0) ncol = 0;
                mbar_arrive_expect_tx(&zfull[warp], (uint32_t)(ncol * nin) * (uint32_t)sizeof(c128));
            }
            __syncwarp();
            if (issuer)
                bulk_g2s(Zs + lane * BT_LDZ, a.Z + (int64_t)mycol * a.ldz + R0 + BT_WR, (uint32_t)nin * (uint32_t)sizeof(c128),
                         &zfull[warp]);
        }
        if constexpr (NSUB > 2) bt_apply_step<GS, (NSUB > 2 ? NSUB - 2 : 0), (NSUB > 2 ? 1 : 0)>(Vs, Qs, Ts, zr, zi, g, t, nrows < BT_WR, nrows);
        if (warp == 0) produce();                 // stage it + STAGES - 1
        if constexpr (NSUB > 1) bt_apply_step<GS, 0, 0>(Vs, Qs, Ts, zr, zi, g, t, nrows < BT_WR, nrows);
        __syncwarp();
        if (lane == 0) mbar_arrive(&empty[slot]);
        if (last) {
            // last step of the unit: store the whole window (generic stores), then publish the unit as complete
#pragma unroll
            for (int p = 0; p < BT_NBLK; ++p)
#pragma unroll
                for (int e = 0; e < 2; ++e) {
                    const int w = 8 * p + 2 * t + e;
                    if (colok && w < nrows) Zc[R0 + w] = cmake(zr[p][e], zi[p][e]);
                }
            if (lane < 8) bulk_wait<0>();
            __syncwarp();
            if (lane == 0) bt_st_release(myprog, hh.k + 1);
            __syncwarp();
        } else {
            // exchange through the staging tile: every lane takes its incoming element and leaves the finished
            // one at the same address; then the 64 finished rows leave by one bulk store per column
            if (nin > 0) {
                mbar_wait(&zfull[warp], zphase);
                zphase ^= 1;
            } else {
                if (lane < 8) bulk_wait_read<0>();                     // no prefetch this step: the tile may still be read
                __syncwarp();
            }
            c128 vin[8][2];
#pragma unroll
            for (int p = 0; p < 8; ++p)
#pragma unroll
                for (int e = 0; e < 2; ++e) {
                    const int w = 8 * p + 2 * t + e;
                    c128* q = Zs + g * BT_LDZ + w;
                    vin[p][e] = (w < nin) ? *q : cmake(0.0, 0.0);
                    *q = cmake(zr[p][e], zi[p][e]);
                }
#pragma unroll
            for (int p = 0; p < BT_NBLK - 8; ++p)
#pragma unroll
                for (int e = 0; e < 2; ++e) { zr[p][e] = zr[p + 8][e]; zi[p][e] = zi[p + 8][e]; }
#pragma unroll
            for (int p = 0; p < 8; ++p)
#pragma unroll
                for (int e = 0; e < 2; ++e) {
                    zr[BT_NBLK - 8 + p][e] = colok ? vin[p][e].x : 0.0;
                    zi[BT_NBLK - 8 + p][e] = colok ? vin[p][e].y : 0.0;
                }
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");     // the tile was written by generic stores
            __syncwarp();
            if (issuer) bulk_s2g(a.Z + (int64_t)mycol * a.ldz + R0, Zs + lane * BT_LDZ, BT_B * (uint32_t)sizeof(c128));
            const bool publish = hh.k > 0 && (hh.k & 15) == 0;      // every 16th step: the release fence is not free
            if (lane < 8) {
                bulk_commit();
                if (publish) bulk_wait<1>();                        // the stores of the steps before this one are complete
            }
            __syncwarp();
            // ---- publish the previous step
            if (publish) {
                if (lane == 0) bt_st_release(myprog, hh.k);
                __syncwarp();
            }
        }
    }
}

template <int GS>
static int bt_launch_sweep(eigh_handle_s* h, const BtSweepArgs& a, cudaStream_t s) {
    auto kern = bt_sweep_kernel<GS>;
    {
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bt_smem(GS));
        if (e != cudaSuccess) return 1000 + (int)e;
    }
    int grid = h->num_sms;
    const long long units = (long long)a.npass * a.nslabs;
    if (grid > units) grid = (int)units;
    cudaEventRecord(h->ev_sweep[0], s);
    kern<<<grid, BT_NT, bt_smem(GS), s>>>(a);
    cudaEventRecord(h->ev_sweep[1], s);
    ++h->launches;
    const cudaError_t e = cudaGetLastError();
    return e != cudaSuccess ? 1000 + (int)e : 0;
}

int launch_pass_off(eigh_handle_s* h, cudaStream_t s) {
    const int npass = (int)bt_npass(h->N);
    bt_pass_off_kernel<<<1, 32, 0, s>>>((int)h->N, npass, ws_ptr<int64_t>(h, h->plan.pass_off));
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
    int* prog = reinterpret_cast<int*>(counter + 2);
    c128* Tneg = ws_ptr<c128>(h, pl.btT);
    EIGH_CUDA_OK(cudaMemsetAsync(counter, 0, 16 + (size_t)npass * nslabs * BT_CWARPS * sizeof(int), s));
    bt_pass_off_kernel<<<1, 32, 0, s>>>(N, npass, pass_off);
    const int kmax = (int)bc_kmax(h);
    int gs = h->g;
    if (gs != 8 && gs != 16 && gs != 32) gs = 8;
    const size_t tp_smem = (size_t)(BT_WR * BT_P + 2 * BT_P * (BT_P + 1) + BT_P) * sizeof(c128);
    EIGH_CUDA_OK(cudaFuncSetAttribute(bt_tprep_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)tp_smem));
    bt_tprep_kernel<<<dim3((unsigned)kmax, (unsigned)npass), 128, tp_smem, s>>>(ws_ptr<c128>(h, pl.V2), ws_ptr<c128>(h, pl.tau2),
                                                                           kmax, N, gs, pass_off, Tneg);
    h->launches += 2;
    BtSweepArgs a;
    a.V2q = nullptr;
    if (bt_qplane(gs)) {
        const int64_t nel = v2_total_stages(N) * BT_VS;
        double* V2q = ws_ptr<double>(h, pl.btQ);
        bt_vq_kernel<<<(unsigned)std::min<int64_t>(ceil_div(nel, 256), 148 * 32), 256, 0, s>>>(ws_ptr<c128>(h, pl.V2), V2q, nel);
        ++h->launches;
        a.V2q = V2q;
    }
    a.Z = Z; a.ldz = ldz; a.N = N; a.nev = nev; a.V2 = ws_ptr<c128>(h, pl.V2); a.Tneg = Tneg; a.pass_off = pass_off;
    a.npass = npass; a.nslabs = nslabs; a.unit_counter = counter; a.prog = prog;
    a.chain = h->bt_chain > 0 ? h->bt_chain : 1;      // chains of 2-4 passes cut the HBM traffic of Z but measure 0.4-1.6 % slower
    if (a.chain > npass) a.chain = npass;
    int rc;
    if (gs == 8) rc = bt_launch_sweep<8>(h, a, s);
    else if (gs == 16) rc = bt_launch_sweep<16>(h, a, s);
    else rc = bt_launch_sweep<32>(h, a, s);
    return rc;
}

}  // namespace eigh
