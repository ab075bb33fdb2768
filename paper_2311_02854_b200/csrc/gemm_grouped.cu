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

const TileShape kVariants[NUM_VARIANTS] = {{64, 64}, {128, 64}, {32, 32}, {16, 16}};

namespace {

constexpr int BK = GEMM_BK;
constexpr int KPAD = BK + 4;   // row stride of a k-contiguous tile (20 = 4 mod 16)

__device__ __forceinline__ void cp_async16(uint32_t dst, const void* src, int src_bytes) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;\n" ::"r"(dst), "l"(src), "r"(src_bytes) : "memory");
}
__device__ __forceinline__ void cp_async8(uint32_t dst, const void* src, int src_bytes) {
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8, %2;\n" ::"r"(dst), "l"(src), "r"(src_bytes) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;\n" ::"n"(N) : "memory"); }

__device__ __forceinline__ void dmma884(double& c0, double& c1, double a, double b) {
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
                 : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}

struct StageMeta { double alpha; uint32_t flags; int32_t ksteps; };

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

// Stage one operand tile (MN x BK) of a segment into shared memory.
//   kcontig: global (mn,k) at g + mn*ld + k, shared at mn*KPAD + k
//   else   : global (mn,k) at g + k*ld + mn, shared at k*(BMN+4) + mn
template <int BMN, int NT>
__device__ __forceinline__ void load_operand(uint32_t sdst, const double* __restrict__ g, int ld, bool kcontig, bool vec2,
                                             int mn_lim, int k_lim, int tid) {
    if (kcontig) {
        if (vec2) {
            constexpr int PAIRS = BMN * (BK / 2);
#pragma unroll
            for (int p = tid; p < PAIRS; p += NT) {
                const int mn = p / (BK / 2), k = (p % (BK / 2)) * 2;
                const bool ok = mn < mn_lim && k < k_lim;
                const int bytes = ok ? (k + 1 < k_lim ? 16 : 8) : 0;
                const double* src = ok ? g + (int64_t)mn * ld + k : g;
                cp_async16(sdst + (mn * KPAD + k) * 8, src, bytes);
            }
        } else {
            constexpr int ELEMS = BMN * BK;
#pragma unroll
            for (int p = tid; p < ELEMS; p += NT) {
                const int mn = p / BK, k = p % BK;
                const bool ok = mn < mn_lim && k < k_lim;
                const double* src = ok ? g + (int64_t)mn * ld + k : g;
                cp_async8(sdst + (mn * KPAD + k) * 8, src, ok ? 8 : 0);
            }
        }
    } else {
        constexpr int MPAD = BMN + 4;
        if (vec2) {
            constexpr int PAIRS = BK * (BMN / 2);
#pragma unroll
            for (int p = tid; p < PAIRS; p += NT) {
                const int k = p / (BMN / 2), mn = (p % (BMN / 2)) * 2;
                const bool ok = mn < mn_lim && k < k_lim;
                const int bytes = ok ? (mn + 1 < mn_lim ? 16 : 8) : 0;
                const double* src = ok ? g + (int64_t)k * ld + mn : g;
                cp_async16(sdst + (k * MPAD + mn) * 8, src, bytes);
            }
        } else {
            constexpr int ELEMS = BK * BMN;
#pragma unroll
            for (int p = tid; p < ELEMS; p += NT) {
                const int k = p / BMN, mn = p % BMN;
                const bool ok = mn < mn_lim && k < k_lim;
                const double* src = ok ? g + (int64_t)k * ld + mn : g;
                cp_async8(sdst + (k * MPAD + mn) * 8, src, ok ? 8 : 0);
            }
        }
    }
}

template <int BM, int BN, int WM, int WN, int NST, int MINB>
__global__ void __launch_bounds__(32 * WM * WN, MINB)
grouped_gemm_kernel(const Job* __restrict__ jobs, const Seg* __restrict__ segs, const Tile* __restrict__ tiles,
                    const double* __restrict__ ops, double* __restrict__ xws, const double* __restrict__ psi,
                    double* __restrict__ sigma) {
    constexpr int NT = 32 * WM * WN;
    constexpr int TM = BM / WM, TN = BN / WN;
    constexpr int FM = TM / 8, FN = TN / 8;
    constexpr int A_ELEMS = (BM * KPAD > BK * (BM + 4)) ? BM * KPAD : BK * (BM + 4);
    constexpr int B_ELEMS = (BN * KPAD > BK * (BN + 4)) ? BN * KPAD : BK * (BN + 4);
    constexpr int STAGE_ELEMS = A_ELEMS + B_ELEMS;
    static_assert(FM >= 1 && FN >= 1, "warp tile must be a multiple of 8x8");

    extern __shared__ __align__(16) double smem[];
    __shared__ StageMeta meta[NST];

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int wm0 = (warp / WN) * TM, wn0 = (warp % WN) * TN;
    const int lr = lane >> 2, lc = lane & 3;

    const Tile tile = tiles[blockIdx.x];
    const Job job = jobs[tile.job];
    const int m0 = tile.tm * BM, n0 = tile.tn * BN;
    const int m_lim = job.M - m0, n_lim = job.N - n0;

    // 8x8 fragments of this warp that intersect the matrix
    const int fm_eff = max(0, min(FM, (m_lim - wm0 + 7) >> 3)), fn_eff = max(0, min(FN, (n_lim - wn0 + 7) >> 3));
    const bool full_tile = fm_eff == FM && fn_eff == FN;
    auto space_r = [&](uint32_t sp) -> const double* { return sp == SP_OPS ? ops : (sp == SP_X ? xws : (sp == SP_PSI ? psi : sigma)); };
    double* const c_base = ((job.flags >> JOB_C_SPACE_SHIFT) & 3u) == SP_X ? xws : sigma;

    double acc[FM][FN][2];
#pragma unroll
    for (int i = 0; i < FM; i++)
#pragma unroll
        for (int j = 0; j < FN; j++) acc[i][j][0] = acc[i][j][1] = 0.0;

    // ---- identity-A segments (planner puts them first): acc += alpha * B tile ---------------------
    int seg0 = job.seg_begin;
    for (; seg0 < job.seg_end; seg0++) {
        const Seg s = segs[seg0];
        if (!(s.flags & SEG_A_IDENT)) break;
        const double* b = space_r((s.flags >> SEG_B_SPACE_SHIFT) & 3u) + s.b_off;
#pragma unroll
        for (int i = 0; i < FM; i++) {
            const int r = m0 + wm0 + 8 * i + lr;
#pragma unroll
            for (int j = 0; j < FN; j++) {
                const int c = n0 + wn0 + 8 * j + 2 * lc;
                if (r < job.M) {
                    if (c < job.N) acc[i][j][0] = fma(s.alpha, b[(int64_t)r * s.ldb + c], acc[i][j][0]);
                    if (c + 1 < job.N) acc[i][j][1] = fma(s.alpha, b[(int64_t)r * s.ldb + c + 1], acc[i][j][1]);
                }
            }
        }
    }

    // ---- pipelined GEMM over the remaining segments ------------------------------------------
    const int nstages = job.pad_;
    int lseg = seg0, lk0 = 0;
    Seg ls;
    if (lseg < job.seg_end) ls = segs[lseg];
    const uint32_t smem_u32 = (uint32_t)__cvta_generic_to_shared(smem);

    auto issue = [&](int slot) {
        if (lseg < job.seg_end) {
            const uint32_t sa = smem_u32 + slot * STAGE_ELEMS * 8;
            const uint32_t sb = sa + A_ELEMS * 8;
            const int k_lim = ls.K - lk0;
            const bool a_kc = !(ls.flags & SEG_A_MCONTIG);
            const bool b_kc = (ls.flags & SEG_B_KCONTIG) != 0;
            const double* ga = space_r((ls.flags >> SEG_A_SPACE_SHIFT) & 3u) + ls.a_off +
                               (a_kc ? (int64_t)m0 * ls.lda + lk0 : (int64_t)lk0 * ls.lda + m0);
            const double* gb = space_r((ls.flags >> SEG_B_SPACE_SHIFT) & 3u) + ls.b_off +
                               (b_kc ? (int64_t)n0 * ls.ldb + lk0 : (int64_t)lk0 * ls.ldb + n0);
            load_operand<BM, NT>(sa, ga, ls.lda, a_kc, (ls.flags & SEG_A_VEC2) != 0, m_lim, k_lim, tid);
            load_operand<BN, NT>(sb, gb, ls.ldb, b_kc, (ls.flags & SEG_B_VEC2) != 0, n_lim, k_lim, tid);
            if (tid == 0) {
                meta[slot].alpha = ls.alpha;
                meta[slot].flags = ls.flags;
                meta[slot].ksteps = (min(k_lim, BK) + 3) >> 2;
            }
            lk0 += BK;
            if (lk0 >= ls.K) {
                lk0 = 0;
                lseg++;
                if (lseg < job.seg_end) ls = segs[lseg];
            }
        }
        cp_async_commit();
    };

#pragma unroll
    for (int s = 0; s < NST - 1; s++) issue(s);

    for (int it = 0; it < nstages; it++) {
        cp_async_wait<NST - 2>();
        __syncthreads();
        issue((it + NST - 1) % NST);
        const int slot = it % NST;
        const double* sa = smem + slot * STAGE_ELEMS;
        const double* sb = sa + A_ELEMS;
        const StageMeta mt = meta[slot];
        const bool a_kc = !(mt.flags & SEG_A_MCONTIG);
        const bool b_kc = (mt.flags & SEG_B_KCONTIG) != 0;
        // element (m,k) of A: a_kc ? m*KPAD + k : k*(BM+4) + m ; fragment: m = wm0+8i+lr, k = 4kk+lc
        const int a_sm = a_kc ? KPAD : 1, a_sk = a_kc ? 1 : BM + 4;
        const int b_sn = b_kc ? KPAD : 1, b_sk = b_kc ? 1 : BN + 4;
        const double* pa = sa + (wm0 + lr) * a_sm + lc * a_sk;
        const double* pb = sb + (wn0 + lr) * b_sn + lc * b_sk;
        const int mode = mt.alpha == 1.0 ? 0 : (mt.alpha == -1.0 ? 1 : 2);
        if (full_tile) {
            for (int kk = 0; kk < mt.ksteps; kk++) {
                double af[FM], bf[FN];
#pragma unroll
                for (int i = 0; i < FM; i++) af[i] = pa[8 * i * a_sm + 4 * kk * a_sk];
#pragma unroll
                for (int j = 0; j < FN; j++) bf[j] = pb[8 * j * b_sn + 4 * kk * b_sk];
                if (mode != 0) scale_frags<FM, FN>(af, bf, mode, mt.alpha);
#pragma unroll
                for (int i = 0; i < FM; i++)
#pragma unroll
                    for (int j = 0; j < FN; j++) dmma884(acc[i][j][0], acc[i][j][1], af[i], bf[j]);
            }
        } else {
            // ragged tile: 8x8 fragments that lie entirely outside the matrix are skipped (warp-uniform
            // predicates), so the executed work is padded to multiples of 8, not of the tile size
            for (int kk = 0; kk < mt.ksteps; kk++) {
                double af[FM], bf[FN];
#pragma unroll
                for (int i = 0; i < FM; i++) af[i] = i < fm_eff ? pa[8 * i * a_sm + 4 * kk * a_sk] : 0.0;
#pragma unroll
                for (int j = 0; j < FN; j++) bf[j] = j < fn_eff ? pb[8 * j * b_sn + 4 * kk * b_sk] : 0.0;
                if (mode != 0) scale_frags<FM, FN>(af, bf, mode, mt.alpha);
#pragma unroll
                for (int i = 0; i < FM; i++)
#pragma unroll
                    for (int j = 0; j < FN; j++)
                        if (i < fm_eff && j < fn_eff) dmma884(acc[i][j][0], acc[i][j][1], af[i], bf[j]);
            }
        }
    }
    cp_async_wait<0>();

    // ---- epilogue: C = beta*C + acc ---------------------------------------------------------------
    const bool beta1 = (job.flags & JOB_BETA1) != 0;
    double* c = c_base + job.c_off;
#pragma unroll
    for (int i = 0; i < FM; i++) {
        const int r = m0 + wm0 + 8 * i + lr;
        if (r >= job.M) continue;
#pragma unroll
        for (int j = 0; j < FN; j++) {
            const int col = n0 + wn0 + 8 * j + 2 * lc;
            double* p = c + (int64_t)r * job.ldc + col;
            if (col < job.N) p[0] = beta1 ? p[0] + acc[i][j][0] : acc[i][j][0];
            if (col + 1 < job.N) p[1] = beta1 ? p[1] + acc[i][j][1] : acc[i][j][1];
        }
    }
}

template <int BM, int BN>
constexpr size_t smem_bytes(int nst) {
    return (size_t)nst * 8 *
           (((BM * KPAD > BK * (BM + 4)) ? BM * KPAD : BK * (BM + 4)) + ((BN * KPAD > BK * (BN + 4)) ? BN * KPAD : BK * (BN + 4)));
}

// variant table: must match kVariants
#define V0 grouped_gemm_kernel<64, 64, 2, 2, 3, 3>
#define V1 grouped_gemm_kernel<128, 64, 4, 2, 3, 1>
#define V2 grouped_gemm_kernel<32, 32, 2, 2, 4, 6>
#define V3 grouped_gemm_kernel<16, 16, 1, 1, 4, 16>

}  // namespace

int gemm_init() {
    static bool done = false;
    if (done) return DMRG_OK;
    DMRG_CUDA(cudaFuncSetAttribute(V0, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_bytes<64, 64>(3)));
    DMRG_CUDA(cudaFuncSetAttribute(V1, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_bytes<128, 64>(3)));
    DMRG_CUDA(cudaFuncSetAttribute(V2, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_bytes<32, 32>(4)));
    DMRG_CUDA(cudaFuncSetAttribute(V3, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_bytes<16, 16>(4)));
    done = true;
    return DMRG_OK;
}

int launch_grouped_gemm(int variant, const Job* jobs, const Seg* segs, const Tile* tiles, int64_t ntiles,
                        const double* ops, double* xws, const double* psi, double* sigma, cudaStream_t st) {
    if (ntiles <= 0) return DMRG_OK;
    const unsigned g = (unsigned)ntiles;
    switch (variant) {
        case 0: V0<<<g, 128, smem_bytes<64, 64>(3), st>>>(jobs, segs, tiles, ops, xws, psi, sigma); break;
        case 1: V1<<<g, 256, smem_bytes<128, 64>(3), st>>>(jobs, segs, tiles, ops, xws, psi, sigma); break;
        case 2: V2<<<g, 128, smem_bytes<32, 32>(4), st>>>(jobs, segs, tiles, ops, xws, psi, sigma); break;
        case 3: V3<<<g, 32, smem_bytes<16, 16>(4), st>>>(jobs, segs, tiles, ops, xws, psi, sigma); break;
        default: set_error("launch_grouped_gemm: bad variant %d", variant); return DMRG_EINVAL;
    }
    DMRG_CUDA(cudaGetLastError());
    return DMRG_OK;
}

}  // namespace dmrg
