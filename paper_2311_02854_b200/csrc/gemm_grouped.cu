// Grouped multi-segment FP64 GEMM for sm_100a -- the hot kernel of sigma = H psi.
//
// One launch executes a list of tiles.  Tile (job, tm, tn) computes a BM x BN tile of
//     C_job = beta * C_job + sum_{s in segments(job)} alpha_s * A_s (M x K_s) * B_s (K_s x N)
// walking the job's segments in plan order with FP64 accumulators in registers, so the result is
// bitwise reproducible and needs no atomics.  Both steps of the paper's GEMM pair map onto it:
//   stage 1 (Eq. 11):      X = psi_panel * (O^R)^T           one segment, beta = 0
//   stage 2 + reduction (Eqs. 12-13):   sigma_blk += sum_mu alpha_mu O^L_mu X_mu   many segments, beta = 1
// (the paper runs Eq. 13 as a separate batched GEMV; here it is the K-loop itself).
//
// Arithmetic: DMMA.8x8x4 (PTX mma.sync.aligned.m8n8k4.f64).  tcgen05 has no FP64 kind, so the
// warp-level DMMA is the FP64 tensor path of sm_100a; measured it issues at the full FP64 pipe rate
// (148 SMs x 64 FMA/clk) while needing 4x fewer shared-memory operands than a DFMA register tile.
// Operands are staged global -> shared with cp.async (16-byte when the planner proved alignment,
// 8-byte otherwise) through an NST-deep ring; zero-fill (src-size 0) pads ragged M, N, K tails.
// Either operand may be read transposed: the shared-memory tile keeps the global orientation and
// only the fragment addressing changes, both orientations being bank-conflict free
// (row strides = 4 mod 16 doubles).
#include "common.h"

namespace dmrg {

const TileShape kVariants[NUM_VARIANTS] = {{64, 64}, {128, 128}, {128, 32}, {32, 128}, {32, 32}};

namespace {

constexpr int BK = GEMM_BK;
constexpr int KPAD = BK + 4;   // row stride of a k-contiguous tile (20 = 4 mod 16)

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

struct StageMeta { double alpha; uint32_t flags; int32_t ksteps; };

// ---- mbarrier helpers (shared::cta) ----------------------------------------------------------------
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;\n" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];\n" ::"r"(bar) : "memory");
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

// fold alpha into the smaller fragment set; |alpha| = 1 flips the sign bit on the integer pipe
// instead of spending an FP64 issue slot
template <int FM, int FN>
__device__ __forceinline__ void scale_frags(double (&af)[FM], double (&bf)[FN], int mode, double alpha) {
    if (FM <= FN) {
#pragma unroll
        for (int i = 0; i < FM; i++)
            af[i] = mode == 1 ? __hiloint2double(__double2hiint(af[i]) ^ 0x80000000, __double2loint(af[i])) : af[i] * alpha;
    } else {
#pragma unroll
        for (int j = 0; j < FN; j++)
            bf[j] = mode == 1 ? __hiloint2double(__double2hiint(bf[j]) ^ 0x80000000, __double2loint(bf[j])) : bf[j] * alpha;
    }
}

// predicated cp.async: no instruction is issued when `on` is false
__device__ __forceinline__ void cp_async8_if(uint32_t dst, const void* src, int src_bytes, bool on) {
    asm volatile("{\n.reg .pred p;\nsetp.ne.b32 p, %3, 0;\n@p cp.async.ca.shared.global [%0], [%1], 8, %2;\n}\n" ::"r"(dst), "l"(src),
                 "r"(src_bytes), "r"((int)on) : "memory");
}

// Stage one operand tile (MN x BK) of a segment into shared memory with NT producer threads.
//   kcontig: global (mn,k) at g + mn*ld + k, shared at mn*KPAD + k
//   else   : global (mn,k) at g + k*ld + mn, shared at k*(BMN+4) + mn
// Elements outside [0, mn_lim) x [0, k_lim) are zero-filled (src-size 0); rows >= round_up(mn_lim, 8) and
// k >= round_up(k_lim, 4) are never read by a fragment and are not copied at all.  Each thread keeps one fixed
// position along the contiguous direction and walks the other with a constant pointer stride, so a copy costs
// a 64-bit add, two compares and the LDGSTS -- the producer warp must not be the bottleneck.
template <int BMN, int NT>
__device__ __forceinline__ void load_operand(uint32_t sdst, const double* __restrict__ g, int ld, bool kcontig, bool vec2,
                                             int mn_lim, int k_lim, int tid) {
    const int mn_end = (mn_lim + 7) & ~7, k_end = (k_lim + 3) & ~3;
    if (vec2 && mn_lim >= BMN && k_lim >= BK) {
        // interior stage (full tile, full K slab): no predicates, no zero-fill -- a copy is the LDGSTS and a 64-bit
        // add.  The producer warp is on the critical path; this is the common case.
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
        if (vec2) {
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
            constexpr int RPI = NT / BK, ITERS = BMN / RPI;
            const int r0 = tid / BK, k = tid % BK;
            const int kb = k < k_lim ? 8 : 0;
            const bool lane_on = k < k_end;
            const double* src = g + (int64_t)r0 * ld + k;
            const int64_t step = (int64_t)RPI * ld;
            const uint32_t dst = sdst + (r0 * KPAD + k) * 8;
#pragma unroll
            for (int i = 0; i < ITERS; i++) {
                const int row = r0 + RPI * i;
                const bool in = row < mn_lim;
                cp_async8_if(dst + i * RPI * KPAD * 8, in ? src : g, in ? kb : 0, lane_on && row < mn_end);
                src += step;
            }
        }
    } else {
        constexpr int MPAD = BMN + 4;
        if (vec2) {
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
        } else {
            constexpr int PR = BMN;
            constexpr int SEGS = PR > NT ? PR / NT : 1;
            constexpr int KPI = PR > NT ? 1 : NT / PR;
            const int k0 = tid / PR, mn0 = tid % PR;
#pragma unroll
            for (int sg = 0; sg < SEGS; sg++) {
                const int mn = mn0 + sg * NT;
                const int mb = mn < mn_lim ? 8 : 0;
                const bool lane_on = mn < mn_end;
                const double* src = g + (int64_t)k0 * ld + mn;
                const int64_t step = (int64_t)KPI * ld;
                const uint32_t dst = sdst + (k0 * MPAD + mn) * 8;
#pragma unroll
                for (int i = 0; i < BK / KPI; i++) {
                    const int k = k0 + KPI * i;
                    const bool in = k < k_lim;
                    cp_async8_if(dst + i * KPI * MPAD * 8, in ? src : g, in ? mb : 0, lane_on && k < k_end);
                    src += step;
                }
            }
        }
    }
}

// One pipeline stage of one consumer warp: up to BK/4 k-steps of FMe x FNe DMMA fragments (the top-left part of
// the warp's FM x FN accumulator grid).  With DBUF the fragments of k-step kk+1 are fetched while the DMMAs of
// k-step kk issue (two k-steps per loop trip, so the buffer index is static).
template <int FM, int FN, int FMe, int FNe, bool DBUF>
__device__ __forceinline__ void compute_stage(double (&acc)[FM][FN][2], const double* __restrict__ pa, const double* __restrict__ pb,
                                              int a_sm, int a_sk, int b_sn, int b_sk, int ksteps, int mode, double alpha) {
    static_assert(FM <= 4 && FN <= 4, "ragged-tile dispatch covers up to 4 x 4 fragments per warp");
    auto mma = [&](double (&af)[FMe], double (&bf)[FNe]) {
        if (mode != 0) scale_frags<FMe, FNe>(af, bf, mode, alpha);
#pragma unroll
        for (int i = 0; i < FMe; i++)
#pragma unroll
            for (int j = 0; j < FNe; j++) dmma884(acc[i][j][0], acc[i][j][1], af[i], bf[j]);
    };
    if (DBUF) {
        uint32_t a_addr = (uint32_t)__cvta_generic_to_shared(pa), b_addr = (uint32_t)__cvta_generic_to_shared(pb);
        const uint32_t a_rs = 64u * a_sm, b_rs = 64u * b_sn, a_ks = 32u * a_sk, b_ks = 32u * b_sk;
        auto loadu = [&](double (&af)[FMe], double (&bf)[FNe]) {
#pragma unroll
            for (int i = 0; i < FMe; i++) af[i] = lds64(a_addr + i * a_rs);
#pragma unroll
            for (int j = 0; j < FNe; j++) bf[j] = lds64(b_addr + j * b_rs);
            a_addr += a_ks;
            b_addr += b_ks;
        };
        double a0[FMe], b0[FNe], a1[FMe], b1[FNe];
        loadu(a0, b0);
#pragma unroll 1
        for (int kk = 0; kk < ksteps; kk += 2) {
            const bool two = kk + 1 < ksteps;
            if (two) loadu(a1, b1);
            mma(a0, b0);
            if (two) {
                if (kk + 2 < ksteps) loadu(a0, b0);
                mma(a1, b1);
            }
        }
    } else {
        // 32-bit shared addresses advanced by a constant per k-step: the k-loop holds no address arithmetic beyond
        // the fragment offsets (indexing by kk made ptxas rematerialise lane ids and reload spilled bases per k-step)
        uint32_t a_addr = (uint32_t)__cvta_generic_to_shared(pa), b_addr = (uint32_t)__cvta_generic_to_shared(pb);
        const uint32_t a_rs = 64u * a_sm, b_rs = 64u * b_sn, a_ks = 32u * a_sk, b_ks = 32u * b_sk;
        const uint32_t a_end = a_addr + ksteps * a_ks;
#pragma unroll 1
        for (; a_addr != a_end; a_addr += a_ks, b_addr += b_ks) {
            double a0[FMe], b0[FNe];
#pragma unroll
            for (int i = 0; i < FMe; i++) a0[i] = lds64(a_addr + i * a_rs);
#pragma unroll
            for (int j = 0; j < FNe; j++) b0[j] = lds64(b_addr + j * b_rs);
            mma(a0, b0);
        }
    }
}

struct ConsumerCtx {
    const Job* job; const Seg* segs; const double* ops; double* xws; const double* psi; double* sigma;
    const double* smem; const StageMeta* meta; uint32_t full_u32, empty_u32;
    int m0, n0, m_lim, n_lim, nstages, lane, wm0, wn0, fm_eff, fn_eff;
};

// Everything one consumer warp does for one tile, with FMe x FNe accumulator fragments (<= the 4 x 4 of a 32x32
// warp tile): identity-A segments, the mbarrier-paced main loop, the epilogue.  Fragments (i, j) with
// i >= fm_eff or j >= fn_eff (a warp ragged in both directions keeps all its columns) are computed on
// zero-filled or neighbouring data and never stored.
template <int BM, int BN, int NST, int FMe, int FNe, bool DBUF>
__device__ __forceinline__ void consumer_body(const ConsumerCtx& cx) {
    constexpr int A_ELEMS = (BM * KPAD > BK * (BM + 4)) ? BM * KPAD : BK * (BM + 4);
    constexpr int B_ELEMS = (BN * KPAD > BK * (BN + 4)) ? BN * KPAD : BK * (BN + 4);
    constexpr int STAGE_ELEMS = A_ELEMS + B_ELEMS;
    const Job& job = *cx.job;
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
    for (int sg = job.seg_begin; sg < job.seg_end; sg++) {
        const Seg s = cx.segs[sg];
        if (!(s.flags & SEG_A_IDENT)) break;
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
    for (int it = 0; it < cx.nstages; it++) {
        const int slot = it % NST;
        mbar_wait(cx.full_u32 + 8 * slot, (it / NST) & 1);
        if (any_frag) {
            const double* sa = cx.smem + slot * STAGE_ELEMS;
            const double* sb = sa + A_ELEMS;
            const StageMeta mt = cx.meta[slot];
            const bool a_kc = !(mt.flags & SEG_A_MCONTIG);
            const bool b_kc = (mt.flags & SEG_B_KCONTIG) != 0;
            // element (m,k) of A: a_kc ? m*KPAD + k : k*(BM+4) + m ; fragment: m = wm0+8i+lr, k = 4kk+lc
            const int a_sm = a_kc ? KPAD : 1, a_sk = a_kc ? 1 : BM + 4;
            const int b_sn = b_kc ? KPAD : 1, b_sk = b_kc ? 1 : BN + 4;
            const double* pa = sa + (wm0 + lr) * a_sm + lc * a_sk;
            const double* pb = sb + (wn0 + lr) * b_sn + lc * b_sk;
            const int mode = (mt.flags & SEG_ALPHA_ONE) ? 0 : ((mt.flags & SEG_ALPHA_NEG) ? 1 : 2);   // integer test: no FP64-pipe DSETP
            compute_stage<FMe, FNe, FMe, FNe, DBUF>(acc, pa, pb, a_sm, a_sk, b_sn, b_sk, mt.ksteps, mode, mt.alpha);
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

// Warp-specialised kernel.  Warps 0 .. WM*WN-1 are CONSUMERS (LDS + DMMA only, one TM x TN warp tile
// each); the last warp is the PRODUCER, which walks the job's segment list and issues every cp.async.
// The two sides meet only through per-stage mbarriers (full: 32 cp.async-completion arrivals + 1
// release arrival that publishes the stage metadata; empty: one arrival per consumer warp), so there
// is no CTA-wide barrier in the main loop and the consumer warps drift freely against each other.
template <int BM, int BN, int WM, int WN, int NST, int NPW, int MAXREG, bool DBUF>
__global__ void __launch_bounds__(32 * (WM * WN + NPW)) __maxnreg__(MAXREG)
grouped_gemm_kernel(const Job* __restrict__ jobs, const Seg* __restrict__ segs, const Tile* __restrict__ tiles,
                    const double* __restrict__ ops, double* __restrict__ xws, const double* __restrict__ psi,
                    double* __restrict__ sigma) {
    constexpr int NCW = WM * WN;   // consumer warps
    constexpr int TM = BM / WM, TN = BN / WN;
    constexpr int FM = TM / 8, FN = TN / 8;
    constexpr int A_ELEMS = (BM * KPAD > BK * (BM + 4)) ? BM * KPAD : BK * (BM + 4);
    constexpr int B_ELEMS = (BN * KPAD > BK * (BN + 4)) ? BN * KPAD : BK * (BN + 4);
    constexpr int STAGE_ELEMS = A_ELEMS + B_ELEMS;
    static_assert(FM >= 1 && FN >= 1, "warp tile must be a multiple of 8x8");

    extern __shared__ __align__(16) double smem[];
    __shared__ StageMeta meta[NST];
    __shared__ __align__(8) uint64_t bar_full[NST], bar_empty[NST];

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;

    const Tile tile = tiles[blockIdx.x];
    if (tile.job < 0) return;   // padding of a thread-block cluster (whole CTA leaves before any barrier)
    const Job job = jobs[tile.job];
    const int m0 = tile.m0, n0 = tile.n0;
    const int m_lim = tile.rows, n_lim = tile.cols;   // <= BM, BN and inside the matrix (planner)
    const int nstages = job.nstages;
    auto space_r = [&](uint32_t sp) -> const double* { return sp == SP_OPS ? ops : (sp == SP_X ? xws : (sp == SP_PSI ? psi : sigma)); };

    const uint32_t full_u32 = (uint32_t)__cvta_generic_to_shared(bar_full);
    const uint32_t empty_u32 = (uint32_t)__cvta_generic_to_shared(bar_empty);
    if (tid == 0) {
#pragma unroll
        for (int s = 0; s < NST; s++) {
            mbar_init(full_u32 + 8 * s, 32 * NPW + 1);
            mbar_init(empty_u32 + 8 * s, NCW);
        }
    }
    __syncthreads();   // the only CTA-wide barrier

    if (warp >= NCW) {
        // =============================== producer warp(s) ============================================
        // NPW == 1: one warp stages A and B; NPW == 2 / 4: the first half of the producer warps stages A, the second half B
        const int pw = warp - NCW;
        int lseg = job.seg_begin;
        while (lseg < job.seg_end && (segs[lseg].flags & SEG_A_IDENT)) lseg++;   // identity segments need no staging
        if (lseg >= job.seg_end) return;
        Seg ls = segs[lseg];
        int lk0 = 0;
        const uint32_t smem_u32 = (uint32_t)__cvta_generic_to_shared(smem);
        for (int it = 0; it < nstages; it++) {
            const int slot = it % NST;
            if (it >= NST) mbar_wait(empty_u32 + 8 * slot, ((it / NST) & 1) ^ 1);
            const uint32_t sa = smem_u32 + slot * STAGE_ELEMS * 8;
            const uint32_t sb = sa + A_ELEMS * 8;
            const int k_lim = ls.K - lk0;
            const bool a_kc = !(ls.flags & SEG_A_MCONTIG);
            const bool b_kc = (ls.flags & SEG_B_KCONTIG) != 0;
            const double* ga = space_r((ls.flags >> SEG_A_SPACE_SHIFT) & 3u) + ls.a_off +
                               (a_kc ? (int64_t)m0 * ls.lda + lk0 : (int64_t)lk0 * ls.lda + m0);
            const double* gb = space_r((ls.flags >> SEG_B_SPACE_SHIFT) & 3u) + ls.b_off +
                               (b_kc ? (int64_t)n0 * ls.ldb + lk0 : (int64_t)lk0 * ls.ldb + n0);
            constexpr int HP = NPW > 1 ? NPW / 2 : 1;   // producer warps per operand
            const int ptid = (pw % HP) * 32 + lane;
            if (NPW == 1 || pw < HP) load_operand<BM, 32 * HP>(sa, ga, ls.lda, a_kc, (ls.flags & SEG_A_VEC2) != 0, m_lim, k_lim, ptid);
            if (NPW == 1 || pw >= HP) load_operand<BN, 32 * HP>(sb, gb, ls.ldb, b_kc, (ls.flags & SEG_B_VEC2) != 0, n_lim, k_lim, ptid);
            mbar_arrive_cp_async(full_u32 + 8 * slot);
            if (pw == 0 && lane == 0) {
                meta[slot].alpha = ls.alpha;
                meta[slot].flags = ls.flags;
                meta[slot].ksteps = (min(k_lim, BK) + 3) >> 2;
                mbar_arrive(full_u32 + 8 * slot);   // release: publishes meta[slot]
            }
            lk0 += BK;
            if (lk0 >= ls.K) {
                lk0 = 0;
                lseg++;
                if (lseg < job.seg_end) ls = segs[lseg];
            }
        }
        return;
    }

    // =================================== consumer warps ================================================
    // The tile's 8x8 fragments are dealt out evenly to the WM x WN consumer warps (a 56 x 48 tile gives the
    // 2 x 2 warps 4+3 by 3+3 fragments): the stage buffers couple the warps of a CTA, so the CTA advances at
    // the pace of its most loaded warp.
    ConsumerCtx cx;
    cx.job = &job; cx.segs = segs; cx.ops = ops; cx.xws = xws; cx.psi = psi; cx.sigma = sigma;
    cx.smem = smem; cx.meta = meta; cx.full_u32 = full_u32; cx.empty_u32 = empty_u32;
    cx.m0 = m0; cx.n0 = n0; cx.m_lim = m_lim; cx.n_lim = n_lim; cx.nstages = nstages; cx.lane = lane;
    const int fr_m = (m_lim + 7) >> 3, fr_n = (n_lim + 7) >> 3;
    const int per_m = (fr_m + WM - 1) / WM, per_n = (fr_n + WN - 1) / WN;
    cx.wm0 = (warp / WN) * per_m * 8; cx.wn0 = (warp % WN) * per_n * 8;
    cx.fm_eff = max(0, min(per_m, fr_m - (warp / WN) * per_m));
    cx.fn_eff = max(0, min(per_n, fr_n - (warp % WN) * per_n));
    // The whole consumer body (accumulators, main loop, epilogue) is specialised on the number of fragment rows
    // OR columns of this warp, so a partly filled tile costs in proportion to its fragments.  (Specialising on
    // both counts at once made ptxas spill; a warp ragged in both directions pads its columns to the warp tile.)
    if (cx.fm_eff == FM || cx.fm_eff == 0) {
        switch (cx.fn_eff) {
            case 1: consumer_body<BM, BN, NST, FM, 1, DBUF>(cx); break;
            case 2: if constexpr (FN >= 2) consumer_body<BM, BN, NST, FM, 2, DBUF>(cx); break;
            case 3: if constexpr (FN >= 3) consumer_body<BM, BN, NST, FM, 3, DBUF>(cx); break;
            default: consumer_body<BM, BN, NST, FM, FN, DBUF>(cx); break;   // full warp tile, or a warp with no fragment
        }
    } else {
        switch (cx.fm_eff) {
            case 1: consumer_body<BM, BN, NST, 1, FN, DBUF>(cx); break;
            case 2: if constexpr (FM >= 2) consumer_body<BM, BN, NST, 2, FN, DBUF>(cx); break;
            default: if constexpr (FM >= 3) consumer_body<BM, BN, NST, 3, FN, DBUF>(cx); break;
        }
    }
}

template <int BM, int BN>
constexpr size_t smem_bytes(int nst) {
    return (size_t)nst * 8 *
           (((BM * KPAD > BK * (BM + 4)) ? BM * KPAD : BK * (BM + 4)) + ((BN * KPAD > BK * (BN + 4)) ? BN * KPAD : BK * (BN + 4)));
}

// variant table: must match kVariants.  <BM, BN, consumer warps M x N, stages, producer warps, register cap, double-buffered fragments>
// Every variant uses 32x32 warp tiles (16 DMMA per 8 LDS.64 per k-step).  V0 was tuned on the B200 (macros kept
// for re-tuning).  Default: BK = 32, 2 stages (72 KB), 128 registers, no spills -> 3 CTAs/SM: half the mbarrier
// round trips per flop of BK = 16.  Measured against BK = 16 / 2 stages / 96 registers / 4 CTAs/SM: cfg 5 +1.7 %,
// cfg 3 +1.0 %, cfg 4 -1.6 %, cfg 2 -2.2 %.  BK = 16 with 3 stages x 128 registers (3 CTAs/SM) lost 4-11 %, 4 stages
// (2 CTAs/SM) and a second producer warp ~10 %, double-buffered fragments at BK = 32 1-5 %.
#ifndef V0_NST
#define V0_NST 2
#endif
#ifndef V0_REG
#define V0_REG 128
#endif
#ifndef V0_DBUF
#define V0_DBUF false
#endif
#ifndef V0_NPW
#define V0_NPW 1
#endif
constexpr int V1_NST = BK >= 32 ? 2 : 4;   // 128x128 stages must fit 227 KB
#define V0 grouped_gemm_kernel<64, 64, 2, 2, V0_NST, V0_NPW, V0_REG, V0_DBUF>
#define V1 grouped_gemm_kernel<128, 128, 4, 4, V1_NST, 4, 96, false>    // large blocks, least operand traffic, 1 CTA/SM
#define V2 grouped_gemm_kernel<128, 32, 4, 1, 3, 1, 128, true>     // skinny N (stage 1 with a small R' sector)
#define V3 grouped_gemm_kernel<32, 128, 1, 4, 3, 1, 128, true>     // skinny M
#define V4 grouped_gemm_kernel<32, 32, 1, 1, 4, 1, 128, true>      // tiny blocks: one consumer warp
constexpr int V0_T = 32 * (4 + V0_NPW), V1_T = 640, V2_T = 160, V3_T = 160, V4_T = 64;
constexpr size_t V0_S = smem_bytes<64, 64>(V0_NST), V1_S = smem_bytes<128, 128>(V1_NST), V2_S = smem_bytes<128, 32>(3), V3_S = smem_bytes<32, 128>(3),
                 V4_S = smem_bytes<32, 32>(4);

}  // namespace

int gemm_init() {
    static bool done = false;
    if (done) return DMRG_OK;
    DMRG_CUDA(cudaFuncSetAttribute(V0, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)V0_S));
    DMRG_CUDA(cudaFuncSetAttribute(V1, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)V1_S));
    DMRG_CUDA(cudaFuncSetAttribute(V2, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)V2_S));
    DMRG_CUDA(cudaFuncSetAttribute(V3, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)V3_S));
    DMRG_CUDA(cudaFuncSetAttribute(V4, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)V4_S));
    done = true;
    return DMRG_OK;
}

template <typename K>
static cudaError_t launch_one(K kernel, unsigned grid, int threads, size_t smem, int cluster, cudaStream_t st, const Job* jobs, const Seg* segs,
                              const Tile* tiles, const double* ops, double* xws, const double* psi, double* sigma) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(grid);
    cfg.blockDim = dim3(threads);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    if (cluster > 1) {
        // sibling tiles of one output block (they share A row panels / B column panels) are launched as one
        // thread-block cluster: co-scheduled, they walk the same K-loop in step and meet in L2
        attr[0].id = cudaLaunchAttributeClusterDimension;
        attr[0].val.clusterDim.x = cluster;
        attr[0].val.clusterDim.y = 1;
        attr[0].val.clusterDim.z = 1;
        cfg.attrs = attr;
        cfg.numAttrs = 1;
    }
    return cudaLaunchKernelEx(&cfg, kernel, jobs, segs, tiles, ops, xws, psi, sigma);
}

int launch_grouped_gemm(int variant, int cluster, const Job* jobs, const Seg* segs, const Tile* tiles, int64_t ntiles,
                        const double* ops, double* xws, const double* psi, double* sigma, cudaStream_t st) {
    if (ntiles <= 0) return DMRG_OK;
    const unsigned g = (unsigned)ntiles;
    cudaError_t e;
    switch (variant) {
        case 0: e = launch_one(V0, g, V0_T, V0_S, cluster, st, jobs, segs, tiles, ops, xws, psi, sigma); break;
        case 1: e = launch_one(V1, g, V1_T, V1_S, cluster, st, jobs, segs, tiles, ops, xws, psi, sigma); break;
        case 2: e = launch_one(V2, g, V2_T, V2_S, cluster, st, jobs, segs, tiles, ops, xws, psi, sigma); break;
        case 3: e = launch_one(V3, g, V3_T, V3_S, cluster, st, jobs, segs, tiles, ops, xws, psi, sigma); break;
        case 4: e = launch_one(V4, g, V4_T, V4_S, cluster, st, jobs, segs, tiles, ops, xws, psi, sigma); break;
        default: set_error("launch_grouped_gemm: bad variant %d", variant); return DMRG_EINVAL;
    }
    if (e != cudaSuccess) { set_error("launch_grouped_gemm: variant %d, %lld tiles, cluster %d: %s", variant, (long long)ntiles, cluster, cudaGetErrorString(e)); return DMRG_ECUDA; }
    return DMRG_OK;
}

}  // namespace dmrg
