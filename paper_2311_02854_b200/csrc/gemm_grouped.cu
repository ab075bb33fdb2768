// Grouped multi-segment FP64 GEMM for sm_100a -- the hot kernel of sigma = H psi.
//
// One launch executes a list of tiles.  Tile (job, tm, tn) computes a BM x BN tile of
//     C_job = beta * C_job + sum_{s in segments(job)} alpha_s * A_s (M x K_s) * B_s (K_s x N)
// walking the job's segments in plan order with FP64 accumulators in registers, so the result is
// bitwise reproducible and needs no atomics.  Both steps of the paper's GEMM pair map onto it:
//   stage 1 (Eq. 11):      X = psi_panel * (O^R)^T           one segment, beta = 0
//   stage 2 + reduction (Eqs. 12-13):   sigma_blk += sum_mu alpha_mu O^L_mu X_mu   many segments, beta = 1
// (the paper runs Eq. 13 as a separate batched GEMV; here it is the K-loop itself), and so does
// the renormalization pair of Eqs. 16-17 with the site tensor in psi's place.
//
// Arithmetic: DMMA.8x8x4 (PTX mma.sync.aligned.m8n8k4.f64).  tcgen05 has no FP64 kind, so the
// warp-level DMMA is the FP64 tensor path of sm_100a; measured it issues at the full FP64 pipe rate
// (148 SMs x 64 FMA/clk) while needing 4x fewer shared-memory operands than a DFMA register tile.
//
// Staging global -> shared (plan option copy_mode):
//   * TMA (default): every operand matrix has a 2-D tensor map (cuTensorMapEncodeTiled, FP64 elements) built by the
//     planner; one elected producer lane issues ONE cp.async.bulk.tensor.2d (SASS UTMALDG) per operand and stage,
//     completion counted in bytes on the stage's "full" mbarrier (expect_tx).  The box is at most 36 x BM (k-contiguous
//     operand) or (BM+4) x 32 (m/n-contiguous) and is shrunk to the operand (a 5 x 300 block is staged as 12 x 64
//     boxes, an 8-column X slice as 12 x 32): the inner box dimension is the extent rounded up to 8 plus 4 padding
//     columns, i.e. = 4 mod 8 doubles, which makes the fragment loads bank-conflict free -- TMA itself writes the
//     padded shared-memory layout, with the pitch travelling in the stage metadata.  Elements outside the operand
//     matrix are zero-filled by the TMA unit (ragged M, N, K tails cost no global traffic); the K tail is
//     additionally masked in registers (compute_stage), which the cp.async path and psi runs rely on.
//   * 16-byte cp.async (LDGSTS) with zero-fill (src-size 0) by all 32 producer lanes: the round-1 path, kept as a
//     selectable alternative (it needs no tensor maps).
// Every operand the planner emits is 16-byte aligned with an even leading dimension (operator blocks and the
// packed R store by construction, psi through the plan's padded copy, X by its even column offsets).
// Either operand may be read transposed: the shared-memory tile keeps the global orientation and only the
// fragment addressing changes, both orientations being bank-conflict free (row strides = 4 mod 16 doubles).
#include "common.h"

namespace dmrg {

const TileShape kVariants[NUM_VARIANTS] = {{64, 64}};

namespace {

constexpr int BK = GEMM_BK;
constexpr int KPAD = BK + 4;   // row stride of a k-contiguous tile (36 = 4 mod 16)

__device__ __forceinline__ void cp_async16(uint32_t dst, const void* src, int src_bytes) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;\n" ::"r"(dst), "l"(src), "r"(src_bytes) : "memory");
}
__device__ __forceinline__ void dmma884(double& c0, double& c1, double a, double b) {
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
                 : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}
__device__ __forceinline__ double lds64(uint32_t addr) {
    double v;
    asm volatile("ld.shared.f64 %0, [%1];\n" : "=d"(v) : "r"(addr));
    return v;
}

struct StageMeta { double alpha; uint32_t flags; int32_t kvalid; uint32_t a_pitch, b_pitch; };   // kvalid: k-columns of this stage inside the segment; pitches in doubles

// ---- mbarrier helpers (shared::cta) ----------------------------------------------------------------
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;\n" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];\n" ::"r"(bar) : "memory");
}
// arrive and add `bytes` to the transaction count the phase waits for (bulk copies complete_tx against it)
__device__ __forceinline__ void mbar_arrive_expect_tx(uint32_t bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;\n" ::"r"(bar), "r"(bytes) : "memory");
}
// arrive on `bar` once all cp.async issued so far by this thread have landed (counts against the init count)
__device__ __forceinline__ void mbar_arrive_cp_async(uint32_t bar) {
    asm volatile("cp.async.mbarrier.arrive.noinc.shared::cta.b64 [%0];\n" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"(bar), "r"(parity) : "memory");
}
// one box of a 2-D tensor map -> shared (dst 128-byte aligned); completion = box bytes on `bar`
__device__ __forceinline__ void tma_load_2d(uint32_t dst, const void* tmap, int c0, int c1, uint32_t bar) {
    asm volatile("cp.async.bulk.tensor.2d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];\n" ::"r"(dst),
                 "l"(tmap), "r"(c0), "r"(c1), "r"(bar) : "memory");
}
__device__ __forceinline__ void tma_prefetch_desc(const void* tmap) {
    asm volatile("prefetch.tensormap [%0];\n" ::"l"(tmap) : "memory");
}

// fold alpha into the A fragments (always A, whatever the fragment counts: the rounding of alpha * a * b must not depend
// on the tile specialisation or the kernel variant); |alpha| = 1 flips the sign bit on the integer pipe instead of spending
// an FP64 issue slot
template <int FM, int FN>
__device__ __forceinline__ void scale_frags(double (&af)[FM], double (&bf)[FN], int mode, double alpha) {
#pragma unroll
    for (int i = 0; i < FM; i++)
        af[i] = mode == 1 ? __hiloint2double(__double2hiint(af[i]) ^ 0x80000000, __double2loint(af[i])) : af[i] * alpha;
}

// ---- producer, cp.async path ----------------------------------------------------------------------------
// Stage one operand tile (MN x BK) of a segment into shared memory with the 32 producer lanes, 16 bytes per copy.
// Elements outside [0, mn_lim) x [0, k_lim) are zero-filled (src-size 0); rows >= round_up(mn_lim, 8) and
// k >= round_up(k_lim, 4) are never read by a fragment and are not copied at all.  Each lane keeps one fixed
// position along the contiguous direction and walks the other with a constant pointer stride.
template <int BMN>
__device__ __forceinline__ void ldgsts_operand(uint32_t sdst, const double* __restrict__ g, int ld, bool kcontig, int mn_lim, int k_lim,
                                               int tid) {
    constexpr int NT = 32;
    const int mn_end = (mn_lim + 7) & ~7, k_end = (k_lim + 3) & ~3;
    if (mn_lim >= BMN && k_lim >= BK) {
        // interior stage (full tile, full K slab): no predicates, no zero-fill
        if (kcontig) {
            constexpr int RPI = NT / (BK / 2), ITERS = BMN / RPI;
            const int r0 = tid / (BK / 2), k = (tid % (BK / 2)) * 2;
            const double* src = g + (int64_t)r0 * ld + k;
            const int64_t step = (int64_t)RPI * ld;
            const uint32_t dst = sdst + (r0 * KPAD + k) * 8;
#pragma unroll
            for (int i = 0; i < ITERS; i++) {
                asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(dst + i * RPI * KPAD * 8), "l"(src) : "memory");
                src += step;
            }
        } else {
            constexpr int MPAD = BMN + 4;
            constexpr int PR = BMN / 2;
            constexpr int SEGS = PR > NT ? PR / NT : 1;
            constexpr int KPI = PR > NT ? 1 : NT / PR;
            const int k0 = tid / PR, mn0 = (tid % PR) * 2;
#pragma unroll
            for (int sg = 0; sg < SEGS; sg++) {
                const int mn = mn0 + sg * NT * 2;
                const double* src = g + (int64_t)k0 * ld + mn;
                const int64_t step = (int64_t)KPI * ld;
                const uint32_t dst = sdst + (k0 * MPAD + mn) * 8;
#pragma unroll
                for (int i = 0; i < BK / KPI; i++) {
                    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(dst + i * KPI * MPAD * 8), "l"(src) : "memory");
                    src += step;
                }
            }
        }
        return;
    }
    if (kcontig) {
        // ragged stage: this lane's rows r0, r0+RPI, ...: full copies (kb bytes of the row's K slab) while the row
        // is inside the matrix, then zero-fill up to the next multiple of 8 rows; loops are bounded by the row
        // counts, so a ragged tile costs the producer in proportion to its rows
        constexpr int RPI = NT / (BK / 2);
        const int r0 = tid / (BK / 2), k = (tid % (BK / 2)) * 2;
        const int kb = k + 1 < k_lim ? 16 : (k < k_lim ? 8 : 0);
        if (k < k_end) {
            const int n_in = mn_lim > r0 ? (mn_lim - r0 + RPI - 1) / RPI : 0;
            const int n_all = mn_end > r0 ? (mn_end - r0 + RPI - 1) / RPI : 0;
            const double* src = g + (int64_t)r0 * ld + k;
            const int64_t step = (int64_t)RPI * ld;
            uint32_t dst = sdst + (r0 * KPAD + k) * 8;
#pragma unroll 4
            for (int i = 0; i < n_in; i++) {
                cp_async16(dst, src, kb);
                src += step;
                dst += RPI * KPAD * 8;
            }
            for (int i = n_in; i < n_all; i++) {
                cp_async16(dst, g, 0);
                dst += RPI * KPAD * 8;
            }
        }
    } else {
        constexpr int MPAD = BMN + 4;
        constexpr int PR = BMN / 2;                              // 16-byte pairs per k-row
        constexpr int SEGS = PR > NT ? PR / NT : 1;              // passes needed to cover one k-row
        constexpr int KPI = PR > NT ? 1 : NT / PR;               // k-rows per pass
        const int k0 = tid / PR, mn0 = (tid % PR) * 2;
        const int n_in = k_lim > k0 ? min(BK / KPI, (k_lim - k0 + KPI - 1) / KPI) : 0;      // k-rows inside the segment
        const int n_all = k_end > k0 ? min(BK / KPI, (k_end - k0 + KPI - 1) / KPI) : 0;     // ... up to the next multiple of 4
#pragma unroll
        for (int sg = 0; sg < SEGS; sg++) {
            const int mn = mn0 + sg * NT * 2;
            if (mn >= mn_end) continue;
            const int mb = mn + 1 < mn_lim ? 16 : (mn < mn_lim ? 8 : 0);
            const double* src = g + (int64_t)k0 * ld + mn;
            const int64_t step = (int64_t)KPI * ld;
            uint32_t dst = sdst + (k0 * MPAD + mn) * 8;
#pragma unroll 4
            for (int i = 0; i < n_in; i++) {
                cp_async16(dst, mb ? src : g, mb);
                src += step;
                dst += KPI * MPAD * 8;
            }
            for (int i = n_in; i < n_all; i++) {
                cp_async16(dst, g, 0);
                dst += KPI * MPAD * 8;
            }
        }
    }
}

// One pipeline stage of one consumer warp: the k-steps of FMe x FNe DMMA fragments covering `kvalid` k-columns.
// The fragments of the last k-step are masked in registers beyond kvalid (lane lc holds k = 4 kk + lc), so the
// shared-memory tile needs no zero K padding.
template <int FMe, int FNe>
__device__ __forceinline__ void compute_stage(double (&acc)[FMe][FNe][2], uint32_t a_addr, uint32_t b_addr, uint32_t a_rs, uint32_t b_rs,
                                              uint32_t a_ks, uint32_t b_ks, int kvalid, int lc, int mode, double alpha) {
    static_assert(FMe <= 4 && FNe <= 4, "ragged-tile dispatch covers up to 4 x 4 fragments per warp");
    auto mma = [&](double (&af)[FMe], double (&bf)[FNe]) {
        if (mode != 0) scale_frags<FMe, FNe>(af, bf, mode, alpha);
#pragma unroll
        for (int i = 0; i < FMe; i++)
#pragma unroll
            for (int j = 0; j < FNe; j++) dmma884(acc[i][j][0], acc[i][j][1], af[i], bf[j]);
    };
    // 32-bit shared addresses advanced by a constant per k-step: the k-loop holds no address arithmetic beyond
    // the fragment offsets (indexing by kk made ptxas rematerialise lane ids and reload spilled bases per k-step)
    const int ksteps = (kvalid + 3) >> 2;
    const int tail = kvalid - 4 * (ksteps - 1);            // valid k-columns of the last k-step: 1..4
    const uint32_t a_end = a_addr + (uint32_t)(tail == 4 ? ksteps : ksteps - 1) * a_ks;
#pragma unroll 1
    for (; a_addr != a_end; a_addr += a_ks, b_addr += b_ks) {
        double a0[FMe], b0[FNe];
#pragma unroll
        for (int i = 0; i < FMe; i++) a0[i] = lds64(a_addr + i * a_rs);
#pragma unroll
        for (int j = 0; j < FNe; j++) b0[j] = lds64(b_addr + j * b_rs);
        mma(a0, b0);
    }
    if (tail != 4) {
        double a0[FMe], b0[FNe];
        const bool keep = lc < tail;
#pragma unroll
        for (int i = 0; i < FMe; i++) { const double v = lds64(a_addr + i * a_rs); a0[i] = keep ? v : 0.0; }
#pragma unroll
        for (int j = 0; j < FNe; j++) { const double v = lds64(b_addr + j * b_rs); b0[j] = keep ? v : 0.0; }
        mma(a0, b0);
    }
}

struct ConsumerCtx {
    const TileDesc* td; const Seg* segs; const double* ops; double* xws; const double* psi; double* sigma;
    uint32_t smem_u32; const StageMeta* meta; uint32_t full_u32, empty_u32;
    int m0, n0, m_lim, n_lim, nstages, lane, wm0, wn0, fm_eff, fn_eff;
    int it0;   // ring position of this sub-tile's first stage (the ring runs on across the sub-tiles of a CTA)
};

// Everything one consumer warp does for one tile, with FMe x FNe accumulator fragments (<= the 4 x 4 of a 32x32
// warp tile): identity-A segments, the mbarrier-paced main loop, the epilogue.  FMe x FNe = the warp's fragment
// counts (fm_eff, fn_eff), except for a warp without fragments, which runs the 1 x 1 body with any_frag = false.
template <int BM, int BN, int NST, int FMe, int FNe>
__device__ __forceinline__ void consumer_body(const ConsumerCtx& cx) {
    constexpr int A_ELEMS = (BM * KPAD > BK * (BM + 4)) ? BM * KPAD : BK * (BM + 4);
    constexpr int B_ELEMS = (BN * KPAD > BK * (BN + 4)) ? BN * KPAD : BK * (BN + 4);
    constexpr int STAGE_ELEMS = A_ELEMS + B_ELEMS;
    const TileDesc& job = *cx.td;
    const int lane = cx.lane, lr = lane >> 2, lc = lane & 3;
    const int m0 = cx.m0, n0 = cx.n0, wm0 = cx.wm0, wn0 = cx.wn0;
    const int fm_eff = cx.fm_eff, fn_eff = cx.fn_eff;
    const bool any_frag = fm_eff > 0 && fn_eff > 0;
    auto space_r = [&](uint32_t sp) -> const double* { return sp == SP_OPS ? cx.ops : (sp == SP_X ? cx.xws : (sp == SP_PSI ? cx.psi : cx.sigma)); };

    double acc[FMe][FNe][2];
#pragma unroll
    for (int i = 0; i < FMe; i++)
#pragma unroll
        for (int j = 0; j < FNe; j++) acc[i][j][0] = acc[i][j][1] = 0.0;

    // ---- identity-A segments (planner puts them first): acc += alpha * B tile ---------------------
    for (int sg = job.seg_begin; sg < job.seg_gemm; sg++) {
        const Seg s = cx.segs[sg];
        const double* b = space_r((s.flags >> SEG_B_SPACE_SHIFT) & 3u) + s.b_off;
#pragma unroll
        for (int i = 0; i < FMe; i++) {
            const int r = m0 + wm0 + 8 * i + lr;
#pragma unroll
            for (int j = 0; j < FNe; j++) {
                const int c = n0 + wn0 + 8 * j + 2 * lc;
                if (i < fm_eff && j < fn_eff && r < m0 + cx.m_lim) {
                    if (c < n0 + cx.n_lim) acc[i][j][0] = fma(s.alpha, b[(int64_t)r * s.ldb + c], acc[i][j][0]);
                    if (c + 1 < n0 + cx.n_lim) acc[i][j][1] = fma(s.alpha, b[(int64_t)r * s.ldb + c + 1], acc[i][j][1]);
                }
            }
        }
    }

    // ---- main loop: wait for a full stage, LDS + DMMA, release it ---------------------------------
    for (int it = cx.it0; it < cx.it0 + cx.nstages; it++) {
        const int slot = it % NST;
        mbar_wait(cx.full_u32 + 8 * slot, (it / NST) & 1);
        if (any_frag) {
            const uint32_t sa = cx.smem_u32 + (uint32_t)slot * (STAGE_ELEMS * 8);
            const uint32_t sb = sa + A_ELEMS * 8;
            const StageMeta mt = cx.meta[slot];
            const bool a_kc = !(mt.flags & SEG_A_MCONTIG);
            const bool b_kc = (mt.flags & SEG_B_KCONTIG) != 0;
            // element (m,k) of A: a_kc ? m*pitch + k : k*pitch + m ; fragment: m = wm0+8i+lr, k = 4kk+lc
            const int a_sm = a_kc ? (int)mt.a_pitch : 1, a_sk = a_kc ? 1 : (int)mt.a_pitch;
            const int b_sn = b_kc ? (int)mt.b_pitch : 1, b_sk = b_kc ? 1 : (int)mt.b_pitch;
            const uint32_t pa = sa + 8u * (uint32_t)((wm0 + lr) * a_sm + lc * a_sk);
            const uint32_t pb = sb + 8u * (uint32_t)((wn0 + lr) * b_sn + lc * b_sk);
            const int mode = (mt.flags & SEG_ALPHA_ONE) ? 0 : ((mt.flags & SEG_ALPHA_NEG) ? 1 : 2);   // integer test: no FP64-pipe DSETP
            compute_stage<FMe, FNe>(acc, pa, pb, 64u * a_sm, 64u * b_sn, 32u * a_sk, 32u * b_sk, mt.kvalid, lc, mode, mt.alpha);
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(cx.empty_u32 + 8 * slot);
    }

    // ---- epilogue: C = beta*C + acc ---------------------------------------------------------------
    const bool beta1 = (job.flags & JOB_BETA1) != 0;
    double* c = (((job.flags >> JOB_C_SPACE_SHIFT) & 3u) == SP_X ? cx.xws : cx.sigma) + job.c_off;
#pragma unroll
    for (int i = 0; i < FMe; i++) {
        const int r = m0 + wm0 + 8 * i + lr;
        if (i >= fm_eff || r >= m0 + cx.m_lim) continue;
#pragma unroll
        for (int j = 0; j < FNe; j++) {
            if (j >= fn_eff) continue;
            const int col = n0 + wn0 + 8 * j + 2 * lc;
            double* p = c + (int64_t)r * job.ldc + col;
            if (col + 1 < n0 + cx.n_lim && ((uintptr_t)p & 15) == 0) {   // the lane's pair as one 16-byte access (X, even-ld sigma rows)
                double2 v = make_double2(acc[i][j][0], acc[i][j][1]);
                if (beta1) { const double2 o = *reinterpret_cast<const double2*>(p); v.x += o.x; v.y += o.y; }
                *reinterpret_cast<double2*>(p) = v;
                continue;
            }
            if (col < n0 + cx.n_lim) p[0] = beta1 ? p[0] + acc[i][j][0] : acc[i][j][0];
            if (col + 1 < n0 + cx.n_lim) p[1] = beta1 ? p[1] + acc[i][j][1] : acc[i][j][1];
        }
    }
}

template <int BM, int BN, int NST, int FMe, int FN, int J>
__device__ __forceinline__ void dispatch_cols(const ConsumerCtx& cx) {
    if constexpr (J <= 1) consumer_body<BM, BN, NST, FMe, 1>(cx);
    else {
        if (cx.fn_eff >= J) consumer_body<BM, BN, NST, FMe, J>(cx);
        else dispatch_cols<BM, BN, NST, FMe, FN, J - 1>(cx);
    }
}
template <int BM, int BN, int NST, int FM, int FN, int I>
__device__ __forceinline__ void dispatch_rows(const ConsumerCtx& cx) {
    if constexpr (I <= 1) dispatch_cols<BM, BN, NST, 1, FN, FN>(cx);
    else {
        if (cx.fm_eff >= I) dispatch_cols<BM, BN, NST, I, FN, FN>(cx);
        else dispatch_rows<BM, BN, NST, FM, FN, I - 1>(cx);
    }
}

// Warp-specialised kernel.  Warps 0 .. WM*WN-1 are CONSUMERS (LDS + DMMA only, one TM x TN warp tile
// each); the last warp is the PRODUCER, which walks the job's segment list and stages every operand tile.
// The two sides meet only through per-stage mbarriers (full: one expect_tx arrival of the elected lane + the
// byte counts of the two TMA copies -- or, on the cp.async path, 32 cp.async-completion arrivals + 1 release
// arrival; either way the arrival publishes the stage metadata; empty: one arrival per consumer warp), so
// there is no CTA-wide barrier in the main loop and the consumer warps drift freely against each other.
template <int BM, int BN, int WM, int WN, int NST, int MAXREG, bool RUNS>
__global__ void __launch_bounds__(32 * (WM * WN + 1)) __maxnreg__(MAXREG)
grouped_gemm_kernel(const Seg* __restrict__ segs, const TileDesc* __restrict__ tiles,
                    const double* __restrict__ ops, double* __restrict__ xws, const double* __restrict__ psi,
                    double* __restrict__ sigma, const TensorMap* __restrict__ tmaps, int copy_mode) {
    constexpr int NCW = WM * WN;   // consumer warps
    constexpr int TM = BM / WM, TN = BN / WN;
    constexpr int FM = TM / 8, FN = TN / 8;
    constexpr int A_ELEMS = (BM * KPAD > BK * (BM + 4)) ? BM * KPAD : BK * (BM + 4);
    constexpr int B_ELEMS = (BN * KPAD > BK * (BN + 4)) ? BN * KPAD : BK * (BN + 4);
    constexpr int STAGE_ELEMS = A_ELEMS + B_ELEMS;
    static_assert(FM >= 1 && FN >= 1, "warp tile must be a multiple of 8x8");

    extern __shared__ __align__(128) double smem[];   // TMA destinations: every stage buffer is a multiple of 128 bytes
    __shared__ StageMeta meta[NST];
    __shared__ __align__(8) uint64_t bar_full[NST], bar_empty[NST];

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;

    const TileDesc job = tiles[blockIdx.x];   // the tile and its job: one 64-byte record
    const int n0 = job.n0, n_lim = job.cols;   // <= BN and inside the matrix (planner)
    const int nstages = job.nstages;   // per sub-tile
    // A CTA computes job.reps sub-tiles of BM rows one after the other (same columns, same segment list; all but the last are
    // full): the stage ring runs on across them, so the copies of the next sub-tile's first stages are in flight while the
    // consumers finish and store the current one -- short tiles (stage 1 at small bond dimensions: K = d_R is a few stages)
    // no longer pay a descriptor fetch and a pipeline fill each.
    // (RUNS = false: the instantiation for launches whose tiles are all single, e.g. stage 2 -- the sub-tile loops fold away)
    const int reps = RUNS ? job.reps : 1;
    auto space_r = [&](uint32_t sp) -> const double* { return sp == SP_OPS ? ops : (sp == SP_X ? xws : (sp == SP_PSI ? psi : sigma)); };

    const uint32_t full_u32 = (uint32_t)__cvta_generic_to_shared(bar_full);
    const uint32_t empty_u32 = (uint32_t)__cvta_generic_to_shared(bar_empty);
    const uint32_t smem_u32 = (uint32_t)__cvta_generic_to_shared(smem);
    if (tid == 0) {
#pragma unroll
        for (int s = 0; s < NST; s++) {
            mbar_init(full_u32 + 8 * s, copy_mode == COPY_TMA ? 1 : 32 + 1);
            mbar_init(empty_u32 + 8 * s, NCW);
        }
    }
    __syncthreads();   // the only CTA-wide barrier

    if (warp >= NCW) {
        // =============================== producer warp ==============================================
        int lseg = job.seg_gemm;   // identity segments need no staging
        if (lseg >= job.seg_end) return;
        if (copy_mode == COPY_TMA) {
            if (lane != 0) return;
            tma_prefetch_desc(tmaps + job.a_map0);   // while the segment descriptor is on its way
            tma_prefetch_desc(tmaps + job.b_map0);
        }
        const Seg ls0 = segs[lseg];
        Seg ls = ls0;
        int lk0 = 0;
        if (copy_mode == COPY_TMA) {
            // ---- TMA: one elected lane, two tensor copies per stage ------------------------------------
            for (int it = 0, rp = 0, m0 = job.m0, st = 0; rp < reps; it++) {
                const int slot = it % NST;
                if (it >= NST) mbar_wait(empty_u32 + 8 * slot, ((it / NST) & 1) ^ 1);
                const uint32_t sa = smem_u32 + (uint32_t)slot * (STAGE_ELEMS * 8);
                const uint32_t sb = sa + A_ELEMS * 8;
                const uint32_t bar = full_u32 + 8 * slot;
                const bool a_kc = !(ls.flags & SEG_A_MCONTIG);
                const bool b_kc = (ls.flags & SEG_B_KCONTIG) != 0;
                meta[slot].alpha = ls.alpha;
                meta[slot].flags = ls.flags;
                meta[slot].kvalid = min(ls.K - lk0, BK);
                meta[slot].a_pitch = ls.a_pitch;
                meta[slot].b_pitch = ls.b_pitch;
                mbar_arrive_expect_tx(bar, ls.a_bytes + ls.b_bytes);   // release: publishes meta[slot]
                tma_load_2d(sa, tmaps + ls.a_map, a_kc ? lk0 : m0, a_kc ? ls.a_o0 + m0 : lk0, bar);
                tma_load_2d(sb, tmaps + ls.b_map, b_kc ? lk0 : n0, b_kc ? n0 : lk0, bar);
                lk0 += BK;
                if (lk0 >= ls.K) {
                    lk0 = 0;
                    lseg++;
                    if (lseg < job.seg_end) {
                        ls = segs[lseg];
                        if (lseg + 1 < job.seg_end) {   // descriptor of the segment after this one: hide its fetch latency
                            tma_prefetch_desc(tmaps + segs[lseg + 1].a_map);
                            tma_prefetch_desc(tmaps + segs[lseg + 1].b_map);
                        }
                    }
                }
                if (++st == nstages) {   // next sub-tile: BM rows further down, the segment list again from its start
                    st = 0; rp++; m0 += BM;
                    lseg = job.seg_gemm; ls = ls0; lk0 = 0;
                }
            }
            return;
        }
        for (int it = 0, rp = 0, m0 = job.m0, st = 0; rp < reps; it++) {
            const int m_lim = rp + 1 < reps ? BM : job.rows;
            const int slot = it % NST;
            if (it >= NST) mbar_wait(empty_u32 + 8 * slot, ((it / NST) & 1) ^ 1);
            const uint32_t sa = smem_u32 + (uint32_t)slot * (STAGE_ELEMS * 8);
            const uint32_t sb = sa + A_ELEMS * 8;
            const uint32_t bar = full_u32 + 8 * slot;
            const int k_lim = ls.K - lk0;
            const bool a_kc = !(ls.flags & SEG_A_MCONTIG);
            const bool b_kc = (ls.flags & SEG_B_KCONTIG) != 0;
            const double* ga = space_r((ls.flags >> SEG_A_SPACE_SHIFT) & 3u) + ls.a_off +
                               (a_kc ? (int64_t)m0 * ls.lda + lk0 : (int64_t)lk0 * ls.lda + m0);
            const double* gb = space_r((ls.flags >> SEG_B_SPACE_SHIFT) & 3u) + ls.b_off +
                               (b_kc ? (int64_t)n0 * ls.ldb + lk0 : (int64_t)lk0 * ls.ldb + n0);
            ldgsts_operand<BM>(sa, ga, ls.lda, a_kc, m_lim, k_lim, lane);
            ldgsts_operand<BN>(sb, gb, ls.ldb, b_kc, n_lim, k_lim, lane);
            mbar_arrive_cp_async(bar);
            if (lane == 0) {
                meta[slot].alpha = ls.alpha;
                meta[slot].flags = ls.flags;
                meta[slot].kvalid = min(k_lim, BK);
                meta[slot].a_pitch = a_kc ? KPAD : BM + 4;
                meta[slot].b_pitch = b_kc ? KPAD : BN + 4;
                mbar_arrive(bar);   // release: publishes meta[slot]
            }
            lk0 += BK;
            if (lk0 >= ls.K) {
                lk0 = 0;
                lseg++;
                if (lseg < job.seg_end) ls = segs[lseg];
            }
            if (++st == nstages) {
                st = 0; rp++; m0 += BM;
                lseg = job.seg_gemm; ls = ls0; lk0 = 0;
            }
        }
        return;
    }

    // =================================== consumer warps ================================================
    // The tile's 8x8 fragments are dealt out to the WM x WN consumer warps (a 56 x 48 tile gives the 2 x 2 warps
    // 4+3 by 3+3 fragments): the stage buffers couple the warps of a CTA, so the CTA advances at the pace of its
    // most loaded warp.
    ConsumerCtx cx;
    cx.td = &job; cx.segs = segs; cx.ops = ops; cx.xws = xws; cx.psi = psi; cx.sigma = sigma;
    cx.smem_u32 = smem_u32; cx.meta = meta; cx.full_u32 = full_u32; cx.empty_u32 = empty_u32;
    cx.n0 = n0; cx.n_lim = n_lim; cx.nstages = nstages; cx.lane = lane;
    const int wr = warp / WN, wc = warp % WN;
    const int fr_n = (n_lim + 7) >> 3, base_n = fr_n / WN, rem_n = fr_n % WN;
    cx.wn0 = (wc * base_n + min(wc, rem_n)) * 8;
    cx.fn_eff = base_n + (wc < rem_n ? 1 : 0);
    for (int rp = 0; rp < reps; rp++) {
        const int m_lim = rp + 1 < reps ? BM : job.rows;
        cx.m0 = job.m0 + rp * BM; cx.m_lim = m_lim; cx.it0 = rp * nstages;
        // deal the sub-tile's fragment rows / columns to the WM x WN warps as evenly as possible: the first (fr % W) warp rows get one more
        const int fr_m = (m_lim + 7) >> 3, base_m = fr_m / WM, rem_m = fr_m % WM;
        cx.wm0 = (wr * base_m + min(wr, rem_m)) * 8;
        cx.fm_eff = base_m + (wr < rem_m ? 1 : 0);
        // The whole consumer body (accumulators, main loop, epilogue) is specialised on the warp's fragment rows AND columns, so a
        // partly filled tile costs exactly its 8 x 8 fragments (a warp without fragments still walks the barriers).
        dispatch_rows<BM, BN, NST, FM, FN, FM>(cx);
    }
}

template <int BM, int BN>
constexpr size_t smem_bytes(int nst) {
    return (size_t)nst * 8 *
           (((BM * KPAD > BK * (BM + 4)) ? BM * KPAD : BK * (BM + 4)) + ((BN * KPAD > BK * (BN + 4)) ? BN * KPAD : BK * (BN + 4)));
}

// One tile shape, two instantiations (with / without the loop over a run of M sub-tiles): 64x64 tile, 2x2 consumer warps
// of 32x32 (16 DMMA per 8 LDS.64 per k-step), BK = 32, 2 stages (72 KB), 114 / 128 registers, no spills -> 3 CTAs/SM.  Measured against it: BK = 16 with 2 / 3 / 4
// stages, 3 stages of BK = 32, a second producer warp, double-buffered fragments, 128-wide tiles, 8 consumer warps of
// 16x32 (better only while the consumer body padded ragged warps to whole warp tiles), a byte ring with up to 8 short
// stages in flight: all slower.
#define V0 grouped_gemm_kernel<64, 64, 2, 2, 2, 128, false>
#define V0R grouped_gemm_kernel<64, 64, 2, 2, 2, 128, true>   // tiles may be runs of M sub-tiles (stage 1)
constexpr int V0_T = 32 * 5;
constexpr size_t V0_S = smem_bytes<64, 64>(2);

}  // namespace

int gemm_init() {
    static bool done = false;
    if (done) return DMRG_OK;
    DMRG_CUDA(cudaFuncSetAttribute(V0, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)V0_S));
    DMRG_CUDA(cudaFuncSetAttribute(V0R, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)V0_S));
    done = true;
    return DMRG_OK;
}

int launch_grouped_gemm(int variant, int copy_mode, const Seg* segs, const TileDesc* tiles, int64_t ntiles,
                        const double* ops, double* xws, const double* psi, double* sigma, const TensorMap* tmaps, cudaStream_t st) {
    if (ntiles <= 0) return DMRG_OK;
    const unsigned g = (unsigned)ntiles;
    switch (variant) {
        case 0: V0<<<g, V0_T, V0_S, st>>>(segs, tiles, ops, xws, psi, sigma, tmaps, copy_mode); break;
        case 1: V0R<<<g, V0_T, V0_S, st>>>(segs, tiles, ops, xws, psi, sigma, tmaps, copy_mode); break;
        default: set_error("launch_grouped_gemm: bad variant %d", variant); return DMRG_EINVAL;
    }
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) { set_error("launch_grouped_gemm: variant %d, %lld tiles: %s", variant, (long long)ntiles, cudaGetErrorString(e)); return DMRG_ECUDA; }
    return DMRG_OK;
}

}  // namespace dmrg
