// bulge.cu -- S2: band -> tridiagonal by bulge chasing ("transforming the banded
// matrix into a tridiagonal form"), SURVEY.md 8(a) rows S2 / S2.1.
//
// Sweep j (j = 0..N-2) annihilates column j below the subdiagonal with a Householder reflector of
// length <= b on rows r_0 = j+1.., applies it two-sided to the diagonal block D_0 and from the right
// to the block S_1 below it (creating a bulge), then chases: at iteration k (r_k = j+1+k b) the
// reflector v_k is applied two-sided to D_k = B[r_k:r_k+b, r_k:r_k+b] and from the right to
// S_{k+1} = B[r_k+b:r_k+2b, r_k:r_k+b]; the first column of S_{k+1} defines v_{k+1}, which is applied
// from the left to the other columns of S_{k+1}.  Every block is loaded once and stored once per
// sweep.  The band keeps up to 2b-1 subdiagonals (lower band storage, ldab >= 2b).
//
// Parallelism: one CTA per sweep in flight (persistent grid, sweeps round-robin over CTAs); sweep
// j+1 may run iteration k once sweep j has finished iteration k+1 (progress counters in global
// memory, acquire/release through L2; all band reads bypass L1).  The grid is launched
// cooperatively so that every CTA is resident (the wait chain always ends at a running sweep).
//
// Reflectors (LAPACK zlarfg convention, H = I - tau v v^H, v_0 = 1 stored explicitly) are packed:
// tile-major (eigh_internal.h): v_{j,k}[i] at V2[((pass_off[j/32] + k) 32 + j%32) 64 + i], zero padded;
// tau of (sweep j, step k) at tau2[j kmax + k].
#include <limits.h>

#include "eigh_internal.h"

namespace eigh {

constexpr int BC_B = 64;          // band width handled by this kernel
constexpr int BC_LD = BC_B + 1;   // padded shared-memory leading dimension of the D block
constexpr int BC_NT = 256;
constexpr int BC_NW = BC_NT / 32;
constexpr int BC_NC = BC_B / 4;   // columns per thread
#ifndef BC_POLL_NS
#define BC_POLL_NS 100
#endif

struct BcArgs {
    c128* band; int64_t ldab;
    int N;
    c128* V2;
    const int64_t* pass_off;
    c128* tau2;       // [N][kmax]: tau of reflector (sweep j, step k) at tau2[j*kmax + k]
    int kmax;
    int* progress;    // [N], zero on entry
    int j_begin, j_end;   // sweeps of this launch: j_begin <= j < j_end (sweep j_begin - 1, if any, is complete)
};

// Thread layout of one chase step: warp w owns rows 8w..8w+7 of a 64 x 64 block; lane = rl + 8 q
// owns row r = 8w + rl and the 16 columns c = q + 4 i.  Row reductions (over columns) are two
// xor-shuffles (8, 16); column reductions (over rows) are a reduce-scatter over the rl lanes
// followed by one pass through shared memory across the 8 warps.  A quarter warp (same q, 8
// consecutive rows) touches 128 contiguous bytes of band storage and 8 distinct shared-memory
// bank groups of the odd-stride D tile.
struct BcSmem {
    c128 D[BC_B * BC_LD];        // lower triangle of D_k (cp.async target)
    c128 zpart[BC_NW * BC_B];    // per-warp partial column sums
    c128 vs[BC_B];               // current reflector (zero padded)
    c128 ws[BC_B];               // w = D v
    c128 zs[BC_B];               // conj(tau') vn^H S
    c128 xs[BC_B];               // first column of S (the next reflector's source)
    double red[BC_NW];
    double red2[BC_NW];
};

__device__ __forceinline__ double bc_warp_sum(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}
__device__ __forceinline__ c128 bc_shfl_xor(c128 v, int m) {
    return cmake(__shfl_xor_sync(0xffffffffu, v.x, m), __shfl_xor_sync(0xffffffffu, v.y, m));
}

// LAPACK zlarfg scalars from alpha = x_0 and xnorm2 = sum_{i>=1} |x_i|^2 (every thread evaluates them
// redundantly: no single-thread section).  v_i = s x_i (i >= 1), v_0 = 1, H x = beta e_1.
__device__ __forceinline__ void bc_reflector_scalars(c128 alpha, double xnorm2, c128& tau, c128& s, double& beta) {
    tau = cmake(0.0, 0.0);
    s = cmake(0.0, 0.0);
    beta = alpha.x;
    if (xnorm2 > 0.0 || alpha.y != 0.0) {
        beta = -copysign(sqrt(alpha.x * alpha.x + alpha.y * alpha.y + xnorm2), alpha.x);
        const double ib = 1.0 / beta;
        tau = cmake((beta - alpha.x) * ib, -alpha.y * ib);
        const double dr = alpha.x - beta, di = alpha.y;
        const double iden = 1.0 / (dr * dr + di * di);
        s = cmake(dr * iden, -di * iden);
    }
}

// ---- inter-CTA progress protocol -------------------------------------------------------------
// progress[j] = number of completed chase steps of sweep j (INT_MAX when the sweep is finished).
// Writer: the compute warps issue their band stores and arrive (without blocking) at a named
// barrier; the publisher warp completes that barrier, executes a gpu-scope release fence (which is
// cumulative over the stores ordered before it by the barrier) and stores the counter.  Reader:
// one thread spins with ld.acquire.gpu; the compute-group barrier that follows orders every later
// band load (all of them bypass L1: cp.async.cg / ld.global.cg) after the acquire.
__device__ __forceinline__ int bc_ld_acquire(const int* p) {
    int v;
    asm volatile("ld.acquire.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void bc_st_release(int* p, int v) {
    asm volatile("fence.acq_rel.gpu;\n\tst.relaxed.gpu.global.s32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}
__device__ __forceinline__ void bc_poll(const int* progress, int sweep, int need) {
    if (sweep >= 0)
        while (bc_ld_acquire(progress + sweep) < need) { __nanosleep(BC_POLL_NS); }
}
// named barriers: 1 = compute group (BC_NT threads); 2, 3 = hand-off to the publisher warp (alternating)
__device__ __forceinline__ void bc_sync_compute() { asm volatile("bar.sync 1, %0;" ::"n"(BC_NT) : "memory"); }
__device__ __forceinline__ void bc_handoff_arrive(int odd) {
    if (odd) asm volatile("bar.arrive 3, %0;" ::"n"(BC_NT + 32) : "memory");
    else asm volatile("bar.arrive 2, %0;" ::"n"(BC_NT + 32) : "memory");
}
__device__ __forceinline__ void bc_handoff_wait(int odd) {
    if (odd) asm volatile("bar.sync 3, %0;" ::"n"(BC_NT + 32) : "memory");
    else asm volatile("bar.sync 2, %0;" ::"n"(BC_NT + 32) : "memory");
}

struct BcStepCtx {
    c128* band; int64_t ldab;
    c128* Vj; c128* tau2j;
    int* progress_j;             // progress counter of the current sweep (!PUB variant releases it itself)
    int r, q, rl, lane, warp, tid;
};

// LAPACK zlarfg on a vector spread over the rows (x = element r, zero for r >= len; all four q lanes of
// a row hold it).  Returns v_r.  One compute-group barrier inside.
__device__ __forceinline__ c128 bc_make_reflector(c128 x, const BcStepCtx& t, int len, double* red, c128* x0,
                                                  c128& tau, double& beta) {
    double part = (t.q == 0 && t.r >= 1 && t.r < len) ? cabs2(x) : 0.0;
    part = bc_warp_sum(part);
    if (t.lane == 0) red[t.warp] = part;
    if (t.r == 0 && t.q == 0) *x0 = x;
    bc_sync_compute();
    double xnorm2 = 0.0;
#pragma unroll
    for (int w = 0; w < BC_NW; ++w) xnorm2 += red[w];
    const c128 alpha = *x0;
    c128 s;
    bc_reflector_scalars(alpha, xnorm2, tau, s, beta);
    c128 v = cmake(0.0, 0.0);
    if (t.r < len) v = (t.r == 0) ? cmake(1.0, 0.0) : cmul(s, x);
    return v;
}

// One chase step (sweep j, step k) by the compute group.  FULL: len = len2 = 64 (no edge predicates).
// Returns false when the sweep ended with this step (no S block below).
// PUB: a ninth (publisher) warp takes the release (one thread block per SM, 168 registers per thread); !PUB: thread 0 of the
// compute group releases after a block barrier (two thread blocks of 8 warps per SM, 128 registers per thread: the second
// block hides the latencies of the first -- used while the sweeps are long enough to keep 2 x 148 blocks busy).
template <bool FULL, bool PUB, bool LEAN = !PUB>
__device__ __forceinline__ bool bc_step(BcSmem& sm, const BcStepCtx& t, int r0, int len_, int len2_, int k, c128& tau, int& hb) {
    const int len = FULL ? BC_B : len_, len2 = FULL ? BC_B : len2_;
    const int r = t.r, q = t.q, rl = t.rl;
    c128* const band = t.band;
    const int64_t ldab = t.ldab;
    // ---- D_k: lower triangle, global -> shared (asynchronous, through L2)
#pragma unroll
    for (int it = 0; it < BC_B * BC_B / BC_NT; ++it) {
        const int idx = t.tid + it * BC_NT;
        const int rr = idx & (BC_B - 1), cc = idx >> 6;
        if (rr >= cc && (FULL || rr < len))
            cp_async16(&sm.D[rr + cc * BC_LD], band + (rr - cc) + (int64_t)(r0 + cc) * ldab, 16);
    }
    cp_async_commit();
    // ---- S_{k+1}: rows r0+b+r, cols r0+c -> registers
    c128 sreg[BC_NC];
    {
        const c128* sp = band + (BC_B + r - q) + (int64_t)(r0 + q) * ldab;    // element (r, c = q); next c: + 4 (ldab - 1)
#pragma unroll
        for (int i = 0; i < BC_NC; ++i) {
            sreg[i] = cmake(0.0, 0.0);
            if (FULL || (r < len2 && q + 4 * i < len)) sreg[i] = __ldcg(sp + (int64_t)i * 4 * (ldab - 1));
        }
    }
    cp_async_wait<0>();
    bc_sync_compute();                                   // D landed; vs of this step visible
    // reflector entries of this thread's 16 columns: registers (PUB) or re-read from shared memory at every use (!PUB:
    // 64 registers fewer; a quarter warp reads one address, i.e. a broadcast)
    c128 vcreg[!LEAN ? BC_NC : 1];
    if constexpr (!LEAN) {
#pragma unroll
        for (int i = 0; i < BC_NC; ++i) vcreg[i] = sm.vs[q + 4 * i];
    }
    auto vc = [&](int i) -> c128 { if constexpr (!LEAN) return vcreg[i]; else return sm.vs[q + 4 * i]; };
    const c128 vr = sm.vs[r];
    // ---- the D phase (two-sided update of D_k) and the S phase (right update of S_{k+1}, next reflector) depend
    //      only on (v, tau): their matrix-vector products run in one loop, their block-wide reductions share one
    //      barrier, and the D update is issued next to the z products of the S phase (independent instruction streams)
    const bool has_s = FULL || len2 > 0;
    c128 wr, ur;
    {
        c128 accd[4], accs[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) accd[u] = accs[u] = cmake(0.0, 0.0);
#pragma unroll
        for (int i = 0; i < BC_NC; ++i) {
            const int c = q + 4 * i;
            c128 e = cmake(0.0, 0.0);
            if (FULL || (r < len && c < len)) {
                e = sm.D[c <= r ? r + c * BC_LD : c + r * BC_LD];      // Hermitian D from its lower triangle
                if (c >= r) e.y = (c == r) ? 0.0 : -e.y;
            }
            const c128 vci = vc(i);
            cfma(accd[i & 3], e, vci);
            cfma(accs[i & 3], sreg[i], vci);
        }
        wr = cadd(cadd(accd[0], accd[1]), cadd(accd[2], accd[3]));
        ur = cadd(cadd(accs[0], accs[1]), cadd(accs[2], accs[3]));
    }
    wr = cadd(wr, bc_shfl_xor(wr, 8));
    ur = cadd(ur, bc_shfl_xor(ur, 8));
    wr = cadd(wr, bc_shfl_xor(wr, 16));
    ur = cadd(ur, bc_shfl_xor(ur, 16));
    // S <- S (I - tau v v^H) in registers:  S -= (tau u) v^H
    {
        const c128 tu = cmul(tau, ur);
#pragma unroll
        for (int i = 0; i < BC_NC; ++i) {
            const c128 vci = vc(i);
            sreg[i].x -= tu.x * vci.x + tu.y * vci.y;
            sreg[i].y -= tu.y * vci.x - tu.x * vci.y;
        }
    }
    // partial sums of v^H (D v) and of the next reflector's norm (first column of S, held by the q = 0 lanes)
    const c128 xs0 = cmake(__shfl_sync(0xffffffffu, sreg[0].x, rl), __shfl_sync(0xffffffffu, sreg[0].y, rl));
    {
        double pa = (q == 0) ? vr.x * wr.x + vr.y * wr.y : 0.0;   // Re(conj(v_r) w_r)
        double pn = (q == 0 && r >= 1 && r < len2) ? cabs2(xs0) : 0.0;
        pa = bc_warp_sum(pa);
        pn = bc_warp_sum(pn);
        if (t.lane == 0) { sm.red[t.warp] = pa; sm.red2[t.warp] = pn; }
        if (q == 0) sm.ws[r] = wr;
        if (r == 0 && q == 0) sm.xs[0] = xs0;
    }
    bc_sync_compute();
    // ---- next reflector (zlarfg scalars, redundantly in every thread)
    c128 taun = cmake(0.0, 0.0);
    double betan = 0.0;
    c128 vnr = cmake(0.0, 0.0);
    if (has_s) {
        double xnorm2 = 0.0;
#pragma unroll
        for (int w = 0; w < BC_NW; ++w) xnorm2 += sm.red2[w];
        c128 sc;
        bc_reflector_scalars(sm.xs[0], xnorm2, taun, sc, betan);
        if (r < len2) vnr = (r == 0) ? cmake(1.0, 0.0) : cmul(sc, xs0);
    }
    // ---- D <- D - v y^H - y v^H,  y = tau w - f v, f = 1/2 |tau|^2 (v^H w):
    //      D[r,c] -= (conj(tau) v_r) conj(w_c) + (tau w_r - 2 f v_r) conj(v_c)   (lower triangle, straight to global)
    {
        double vhw = 0.0;
#pragma unroll
        for (int w = 0; w < BC_NW; ++w) vhw += sm.red[w];
        const double f2 = (tau.x * tau.x + tau.y * tau.y) * vhw;
        const c128 pr = cmulc(tau, vr);                    // conj(tau) v_r
        const c128 twr = cmul(tau, wr);
        const c128 qr = cmake(twr.x - f2 * vr.x, twr.y - f2 * vr.y);
        if (FULL || r < len) {
            c128* dp = band + (r - q) + (int64_t)(r0 + q) * ldab;
#pragma unroll
            for (int i = 0; i < BC_NC; ++i) {
                const int c = q + 4 * i;
                if (c <= r) {
                    const c128 wc = sm.ws[c];
                    const c128 vci = vc(i);
                    c128 e = sm.D[r + c * BC_LD];
                    e.x -= pr.x * wc.x + pr.y * wc.y + qr.x * vci.x + qr.y * vci.y;
                    e.y -= pr.y * wc.x - pr.x * wc.y + qr.y * vci.x - qr.x * vci.y;
                    if (c == r) e.y = 0.0;
                    dp[(int64_t)i * 4 * (ldab - 1)] = e;
                }
            }
        }
    }
    // ---- early hand-off.  The next sweep's step k-1 overlaps this step's blocks only in the first column of D_k (stored
    //      above) and in S_{k+1}(0,0) = beta' (stored here); everything else it reads was final one step ago.  So the
    //      release of "step k" is handed to the publisher warp now, and the rest of the step (left update of S_{k+1}, its
    //      stores, the reflector) runs behind it: the lag between consecutive sweeps drops from 2 steps to ~1.6.
    if (has_s && r == 0 && q == 0) band[BC_B + (int64_t)r0 * ldab] = cmake(betan, 0.0);
    if constexpr (PUB) {
        bc_handoff_arrive(hb);
        hb ^= 1;
    } else {
        bc_sync_compute();                                   // every thread's stores of this step are issued
        if (t.tid == 0) bc_st_release(t.progress_j, has_s ? k + 1 : INT_MAX);
    }
    if (!has_s) return false;
    // ---- z_c = vn^H S[:, c]: per-thread products, reduce-scatter over the 8 row lanes, then across warps
    {
        // (the first exchange is folded into the products: 8 partial sums are live instead of 16)
        c128 zp[BC_NC / 2];
        {
            const bool up0 = rl & 1;
#pragma unroll
            for (int i = 0; i < BC_NC / 2; ++i) {
                const c128 a0 = cmulc(vnr, sreg[i]), a1 = cmulc(vnr, sreg[i + BC_NC / 2]);
                zp[i] = cadd(up0 ? a1 : a0, bc_shfl_xor(up0 ? a0 : a1, 1));
            }
        }
#pragma unroll
        for (int st = 1; st < 3; ++st) {
            const int half = BC_NC >> (st + 1);
            const bool up = (rl >> st) & 1;
#pragma unroll
            for (int i = 0; i < half; ++i) {
                const c128 send = up ? zp[i] : zp[i + half];
                const c128 keep = up ? zp[i + half] : zp[i];
                zp[i] = cadd(keep, bc_shfl_xor(send, 1 << st));
            }
        }
        // zp[i'] (i' = 0, 1) is the sum over the warp's rows of column index i = i' + 2 b2 + 4 b1 + 8 b0
        const int ibase = ((rl >> 2) & 1) * 2 + ((rl >> 1) & 1) * 4 + (rl & 1) * 8;
        sm.zpart[t.warp * BC_B + q + 4 * (ibase + 0)] = zp[0];
        sm.zpart[t.warp * BC_B + q + 4 * (ibase + 1)] = zp[1];
    }
    bc_sync_compute();
    if (t.tid < BC_B) {
        c128 z0 = cadd(sm.zpart[0 * BC_B + t.tid], sm.zpart[1 * BC_B + t.tid]);
        c128 z1 = cadd(sm.zpart[2 * BC_B + t.tid], sm.zpart[3 * BC_B + t.tid]);
        c128 z2 = cadd(sm.zpart[4 * BC_B + t.tid], sm.zpart[5 * BC_B + t.tid]);
        c128 z3 = cadd(sm.zpart[6 * BC_B + t.tid], sm.zpart[7 * BC_B + t.tid]);
        sm.zs[t.tid] = cmulc(taun, cadd(cadd(z0, z1), cadd(z2, z3)));        // conj(tau') z_c
    }
    bc_sync_compute();
    // ---- S[:, c] -= vn (conj(tau') z_c) for c >= 1; S[:, 0] = beta' e_1; store S and the reflector
    {
        c128* sp = band + (BC_B + r - q) + (int64_t)(r0 + q) * ldab;
#pragma unroll
        for (int i = 0; i < BC_NC; ++i) {
            const int c = q + 4 * i;
            c128 e = sreg[i];
            if (c == 0) e = (r == 0) ? cmake(betan, 0.0) : cmake(0.0, 0.0);
            else {
                const c128 zc = sm.zs[c];
                e.x -= vnr.x * zc.x - vnr.y * zc.y;
                e.y -= vnr.x * zc.y + vnr.y * zc.x;
            }
            // (0,0) was stored before the hand-off and may already have been updated by the next sweep
            if ((FULL || (r < len2 && c < len)) && !(c == 0 && r == 0)) sp[(int64_t)i * 4 * (ldab - 1)] = e;
        }
    }
    if (q == 0) {
        __stcs(t.Vj + (int64_t)(k + 1) * (32 * BC_B) + r, vnr);  // zero beyond len2; write-once: streaming, keeps the band in L2
        sm.vs[r] = vnr;
    }
    if (t.tid == 0) t.tau2j[k + 1] = taun;
    tau = taun;
    return true;
}

// VAR 0: publisher warp, one block per SM (default).  VAR 1: no publisher, lean registers, two blocks per SM (bc_dual_steps).
// VAR 2: no publisher, one block per SM with the full register file (255 registers, no spills; option bc_variant = 2).
// VAR 3: publisher warp AND the full register file for the compute warps: three warpgroups (8 compute warps, the publisher
//        warp + 3 idle warps); the publisher's warpgroup gives its registers back (setmaxnreg.dec) and the compute
//        warpgroups take them (setmaxnreg.inc 232), so the compute code needs no spills (option bc_variant = 3).
template <int VAR>
__global__ void __launch_bounds__(VAR == 3 ? BC_NT + 128 : VAR == 0 ? BC_NT + 32 : BC_NT, VAR == 1 ? 2 : 1) bulge_chase_kernel(const BcArgs a) {
    constexpr bool PUB = VAR == 0 || VAR == 3, LEAN = VAR == 1;
    extern __shared__ __align__(16) unsigned char bc_raw[];
    BcSmem& sm = *reinterpret_cast<BcSmem*>(bc_raw);

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int N = a.N;

    if (PUB && warp >= BC_NW) {
        // ================= publisher warp: one release per step whose D phase is complete (the previous step is then
        // complete in full), INT_MAX per completed sweep.  (VAR 3: its whole warpgroup first hands its registers back.)
        if constexpr (VAR == 3) {
            asm volatile("setmaxnreg.dec.sync.aligned.u32 32;");
            if (warp > BC_NW) return;
        }
        int hb = 0;
        for (int j = a.j_begin + blockIdx.x; j < a.j_end; j += gridDim.x) {
            for (int k = 0;; ++k) {
                const bool more = N - (j + 1 + k * BC_B + BC_B) > 0;
                bc_handoff_wait(hb);
                hb ^= 1;
                if (lane == 0) bc_st_release(a.progress + j, more ? k + 1 : INT_MAX);
                if (!more) break;
            }
        }
        return;
    }
    if constexpr (VAR == 3) asm volatile("setmaxnreg.inc.sync.aligned.u32 232;");

    BcStepCtx t;
    t.band = a.band; t.ldab = a.ldab;
    t.tid = tid; t.lane = lane; t.warp = warp;
    t.rl = lane & 7; t.q = lane >> 3; t.r = warp * 8 + t.rl;
    const int r = t.r, q = t.q;
    int hb = 0;

    for (int j = a.j_begin + blockIdx.x; j < a.j_end; j += gridDim.x) {
        t.Vj = a.V2 + ((a.pass_off[j >> 5] * 32 + (j & 31)) * BC_B);     // reflector (j, k) at Vj[k * 2048 + i]
        t.tau2j = a.tau2 + (int64_t)j * a.kmax;
        t.progress_j = a.progress + j;
        if (tid == 0) bc_poll(a.progress, j - 1, 2);
        bc_sync_compute();
        // ---- reflector (j, 0) from column j of the band
        c128 tau;
        {
            const int len = min(BC_B, N - 1 - j);
            c128* colj = a.band + (int64_t)j * a.ldab;
            c128 x = cmake(0.0, 0.0);
            if (r < len) x = __ldcg(colj + 1 + r);
            double beta;
            const c128 vr = bc_make_reflector(x, t, len, sm.red2, &sm.xs[0], tau, beta);
            if (q == 0) {
                if (r < len) {
                    colj[1 + r] = (r == 0) ? cmake(beta, 0.0) : cmake(0.0, 0.0);
                }
                __stcs(t.Vj + r, vr);                         // zero beyond len
                sm.vs[r] = vr;
            }
            if (tid == 0) t.tau2j[0] = tau;
        }
        for (int k = 0;; ++k) {
            const int r0 = j + 1 + k * BC_B;
            const int len = min(BC_B, N - r0);
            const int len2 = min(BC_B, N - (r0 + BC_B));
            // (the release of the step is handed to the publisher warp inside bc_step, after the D phase)
            const bool more = (len == BC_B && len2 == BC_B) ? bc_step<true, PUB, LEAN>(sm, t, r0, len, len2, k, tau, hb)
                                                            : bc_step<false, PUB, LEAN>(sm, t, r0, len, len2, k, tau, hb);
            if (!more) break;
            // (one polling thread + a block barrier: eight polling warps measured 8 % slower -- they compete for the L2)
            if (tid == 0) bc_poll(a.progress, j - 1, k + 3);
            bc_sync_compute();
        }
    }
}

// d_i = Re B[i,i]; e_i = |B[i+1,i]| (real by construction); sgn_0 = 1, sgn_{i+1} = sgn_i sign(B[i+1,i]).
__global__ void extract_tridiag_kernel(const c128* __restrict__ band, int64_t ldab, int N, double* __restrict__ d,
                                       double* __restrict__ e, double* __restrict__ sgn) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < N) d[i] = band[(int64_t)i * ldab].x;
    if (i < N - 1) e[i] = fabs(band[1 + (int64_t)i * ldab].x);
    if (i == 0) {
        double s = 1.0;
        sgn[0] = 1.0;
        for (int t = 0; t < N - 1; ++t) {
            if (band[1 + (int64_t)t * ldab].x < 0.0) s = -s;
            sgn[t + 1] = s;
        }
    }
}

// zero the last stage (32 reflectors x 64 elements) of pass blockIdx.x
__global__ void bc_zero_last_stage_kernel(c128* __restrict__ V2, const int64_t* __restrict__ pass_off) {
    const int64_t first = pass_off[blockIdx.x], next = pass_off[blockIdx.x + 1];
    if (next <= first) return;
    c128* st = V2 + (next - 1) * (32 * BC_B);
    for (int i = threadIdx.x; i < 32 * BC_B; i += blockDim.x) st[i] = cmake(0.0, 0.0);
}

int phase_band_to_tridiag(eigh_handle_s* h, c128* band, int64_t ldab, double* d, double* e, cudaStream_t s) {
    const int N = (int)h->N;
    if (h->b != BC_B) return set_err(h, -100, "bulge chasing is built for band width %d", BC_B);
    const WsPlan& pl = h->plan;
    int* progress = ws_ptr<int>(h, pl.bc_progress);
    double* sgn = ws_ptr<double>(h, pl.sgn);
    EIGH_CUDA_OK(cudaMemsetAsync(progress, 0, (size_t)(N + 8) * sizeof(int), s));
    {
        const int rc = launch_pass_off(h, s);
        if (rc) return rc;
    }
    // Reflector slots that no (sweep, step) writes must read as zero.  Sweep j has ceil((N-1-j)/64) steps and a pass of 32
    // sweeps has as many stages as its FIRST sweep has steps, so only the LAST stage of a pass can hold unwritten slots
    // (later sweeps of the pass that are one step shorter, sweeps beyond N-2): 32 KB per pass instead of the whole array.
    if (v2_npass(N) > 0) {
        bc_zero_last_stage_kernel<<<(unsigned)v2_npass(N), 256, 0, s>>>(ws_ptr<c128>(h, pl.V2), ws_ptr<int64_t>(h, pl.pass_off));
        ++h->launches;
    }
    if (N >= 2) {
        const size_t smem = sizeof(BcSmem);
        BcArgs a;
        a.band = band; a.ldab = ldab; a.N = N; a.V2 = ws_ptr<c128>(h, pl.V2); a.progress = progress;
        a.pass_off = ws_ptr<int64_t>(h, pl.pass_off);
        a.tau2 = ws_ptr<c128>(h, pl.tau2); a.kmax = (int)bc_kmax(h);
        // Long sweeps first, with TWO thread blocks per SM (no publisher warp, 128 registers): while a sweep has more than
        // ~2 x (2 x 148) steps every block is busy and the second block of an SM hides the latencies of the first.  The
        // remaining sweeps run with one block per SM (publisher warp, 168 registers), whose single step is faster: there the
        // lag between consecutive sweeps, not the number of blocks, bounds the rate.
        int j_switch = 0;
        if (h->bc_dual_steps > 0) {
            const int64_t js = (int64_t)N - 1 - (int64_t)h->bc_dual_steps * BC_B;
            j_switch = js > 0 ? (int)js : 0;
            if (j_switch > N - 1) j_switch = N - 1;
        }
        void* kargs[] = {(void*)&a};
        if (j_switch > 0) {
            auto kern = bulge_chase_kernel<1>;
            EIGH_CUDA_OK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
            int occ = 0;
            EIGH_CUDA_OK(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kern, BC_NT, smem));
            if (occ < 1) return set_err(h, EIGH_ERR_CUDA, "bulge_chase_kernel<dual> cannot be resident");
            int G = h->num_sms * occ;
            if (h->bc_grid > 0 && h->bc_grid < G) G = h->bc_grid;
            if (G > j_switch) G = j_switch;
            a.j_begin = 0; a.j_end = j_switch;
            EIGH_CUDA_OK(cudaLaunchCooperativeKernel((void*)kern, dim3(G), dim3(BC_NT), kargs, smem, s));
            ++h->launches;
        }
        if (j_switch < N - 1) {
            const int var = h->bc_variant;
            void (*kern)(const BcArgs) = var == 2 ? bulge_chase_kernel<2> : var == 3 ? bulge_chase_kernel<3> : bulge_chase_kernel<0>;
            const int nthreads = var == 2 ? BC_NT : var == 3 ? BC_NT + 128 : BC_NT + 32;
            EIGH_CUDA_OK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
            int occ = 0;
            EIGH_CUDA_OK(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kern, nthreads, smem));
            if (occ < 1) return set_err(h, EIGH_ERR_CUDA, "bulge_chase_kernel cannot be resident");
            int G = h->num_sms * occ;
            if (h->bc_grid > 0 && h->bc_grid < G) G = h->bc_grid;
            if (G > N - 1 - j_switch) G = N - 1 - j_switch;
            a.j_begin = j_switch; a.j_end = N - 1;
            EIGH_CUDA_OK(cudaLaunchCooperativeKernel((void*)kern, dim3(G), dim3(nthreads), kargs, smem, s));
            ++h->launches;
        }
    }
    extract_tridiag_kernel<<<(unsigned)ceil_div(N, 256), 256, 0, s>>>(band, ldab, N, d, e, sgn);
    ++h->launches;
    const cudaError_t ce = cudaGetLastError();
    return ce != cudaSuccess ? 1000 + (int)ce : 0;
}

}  // namespace eigh
