// dmrg_plan_create / dmrg_sigma / dmrg_hdiag.
//
// The planner is the paper's "CPU preprocessing": every term mu of Eq. (5) and every
// combination of symmetry blocks becomes a GEMM pair (Eq. 14).  Differences from the paper's design
// (cublasDgemmBatched per equal-shape group on many streams), chosen for one B200:
//   * stage-1 products X = psi_blk * (O^R_blk)^T are de-duplicated (X depends only on the R block and
//     the psi block, and one-index R operators recur in many terms); because psi is laid out with all
//     blocks of one R sector back to back, consecutive psi blocks are merged along M; and R blocks applied
//     to the same psi rows are merged along N through a plan-owned packed copy (K-contiguous, h.c. uses
//     transposed), so one tall-and-wide GEMM replaces hundreds of small ones;
//   * all contributions to one sigma block are concatenated along K into ONE GEMM whose K-loop walks
//     the (term, input block) pairs in a fixed order -- this is Eq. (13) without a separate reduction
//     kernel and without atomics;
//   * no grouping by equal shape: a single kernel walks a cost-sorted tile list with per-tile shapes.
// Terms are processed in chunks sized so the X intermediates fit the workspace.
#include <algorithm>
#include <array>
#include <atomic>
#include <cmath>
#include <complex>
#include <cstdlib>
#include <new>
#include <thread>
#include <unordered_map>

#include "plan.h"
#include "tmap.h"

namespace dmrg {

static const int SITE_N[4] = {0, 1, 1, 2};
static const int SITE_S[4] = {0, -1, 1, 0};

// Complex plans (dmrg_plan_create_z, spin-orbit Hamiltonians: PAPER.md:97): the complex contraction runs through the
// same real grouped GEMMs.  psi, X and sigma are kept "row-planar" (row l = [re | im], each half padded to an even
// length): stage 1 multiplies such rows (K = both halves) by the real image [[Rre, -Rim], [Rim, Rre]] of the R block
// as used, packed K-contiguous with all real-part rows of a stack before all imaginary-part rows, so X comes out
// row-planar again; read with half the row pitch, a row-planar dL x dR' matrix IS the real 2 dL x dR' matrix whose rows
// 2l, 2l+1 are (re, im) of row l, which is what the interleaved real image of an L block (ops_store.cu) multiplies in
// stage 2 -- M and K double, N stays.  One complex GEMM costs 4 real ones (8 M N K flops), nothing is computed twice.
// A complex coefficient alpha = ar + i ai gives two real tasks: ar into accumulator 0, ai into accumulator 1 (the
// second half of the plan's internal sigma buffer, out_blk + nblk); sigma = acc0 + i acc1 is formed when the
// row-planar result is written out interleaved (sigma_z_finish_kernel).  `zdim` below = 2 for complex plans.
struct Task {
    int32_t term_ord, in_blk, out_blk;
    int32_t l_trans, r_trans;
    int32_t dLi, dLo, dRi, dRo;
    int64_t l_off, r_off;   // device offsets of the operator blocks, -1 = identity
    double alpha;
    int32_t canon;          // 1: counts towards the canonical flops (0: the imaginary-coefficient twin of a complex task)
};

struct XLoc { int64_t off; int32_t ld; };   // X of one task: a slice (origin, row pitch) of a stage-1 job's output matrix

static inline int64_t xkey(int64_t r_off, int r_trans, int in_blk, int64_t nblk) {
    return (r_off * 2 + r_trans) * nblk + in_blk;
}

// Tile variant for an M x N output: one variant today (64x64 tile, 2 x 2 consumer warps).  Since its consumer
// body is specialised on the warp's fragment counts it also handled skinny and tiny outputs better than the
// dedicated 128x32 / 32x128 / 32x32 / 128x128 tiles of round 1 did, which are gone.
static int choose_variant(int /*M*/, int /*N*/) { return 0; }

// fragments a tile costs when every consumer warp is charged the load of the most loaded one (WM x WN warps)
static inline double warp_area(const std::vector<std::pair<int, int>>& cm, const std::vector<std::pair<int, int>>& cn, int v) {
    const int wm = kVariants[v].bm / 32, wn = kVariants[v].bn / 32;
    double a = 0;
    for (auto& m : cm)
        for (auto& n : cn) {
            const int fm = (m.second + 7) / 8, fn = (n.second + 7) / 8;
            a += 64.0 * wm * wn * ((fm + wm - 1) / wm) * ((fn + wn - 1) / wn);
        }
    return a;
}

static inline double frag_area(int M, int N) { return 64.0 * ((M + 7) / 8) * ((N + 7) / 8); }

__global__ void pack_r_kernel(const PackDesc* __restrict__ descs, const double* __restrict__ ops, double* __restrict__ pack);
__global__ void pack_r_z_kernel(const PackDesc* __restrict__ descs, const double* __restrict__ ops, double* __restrict__ pack);

struct TileRec { Tile t; double cost; int64_t key = 0; int32_t bucket = 0; };   // key: secondary launch order inside a cost bucket

constexpr int64_t kPackBase = int64_t(1) << 50;   // marks b_off values that are offsets into the packed R store

// split-K policy of stage 2 (see the comment at its use): the wave count is in units of 592 CTA slots (the sweep of
// DESIGN.md section 9 was taken with 4 resident CTAs per SM; the BK = 32 kernel keeps 3, the unit is kept so that the
// recorded numbers stay comparable)
constexpr double kCtaSlots = 148.0 * 4;

struct PlanPolicy {   // dmrg_plan_options with the defaults filled in
    int64_t workspace_bytes;
    int copy_mode;
    double split_waves, min_split_stages;
    int64_t max_merged_cols;
    bool tile_order;
    int split_small;
    bool release_r_store;
    bool release_staged;   // release_r_store == 2: always park the R side on the host while the pack is filled
    int shard_rank, shard_count;
    int tile_run_stages;   // stage 1: a CTA computes as many consecutive M tiles as it takes to reach this many pipeline stages (<= 8 tiles)
};

static PlanPolicy make_policy(const dmrg_plan_options* o) {
    PlanPolicy p;
    p.workspace_bytes = (o && o->workspace_bytes > 0) ? o->workspace_bytes : (int64_t(8) << 30);
    p.copy_mode = (o && (o->copy_mode == COPY_LDGSTS || o->copy_mode == COPY_TMA)) ? o->copy_mode : COPY_TMA;
    // split-K defaults re-measured on the final round-2 kernel (profiles/r2_summary.md section 6): 100 waves, parts of at least
    // K = 3072 (96 stages): cfg2 -3.7 %, cfg3 -1.0 %, cfg4 -0.5 %, cfg5 -0.4 % against the 200 waves / K = 768 of round 1
    p.split_waves = (o && o->split_waves > 0) ? o->split_waves : 100.0;
    p.min_split_stages = (o && o->min_split_stages > 0) ? (double)o->min_split_stages : 3072.0 / GEMM_BK;
    p.max_merged_cols = (o && o->max_merged_cols >= 64) ? (int64_t)(o->max_merged_cols & ~1) : int64_t(4096);
    p.tile_order = !(o && o->cost_order_only);
    p.split_small = (o && o->split_small > 0) ? o->split_small : 0;
    p.release_r_store = o && o->release_r_store;
    p.release_staged = o && o->release_r_store == 2;
    p.tile_run_stages = (o && o->tile_run_stages > 0) ? o->tile_run_stages : 32;
    p.shard_count = (o && o->shard_count > 1) ? o->shard_count : 1;
    p.shard_rank = (o && o->shard_count > 1) ? o->shard_rank : 0;
    return p;
}

static int plan_build(dmrg_plan* P, const dmrg_term* terms, const double* coef_im, int64_t nterms_in, const double* site_ops_in,
                      const int32_t* site_parity, int32_t nsite, int32_t n_total, int32_t two_sz_total,
                      const PlanPolicy& pol) {
    const bool Z = P->ops->cplx;   // complex plan: site_ops_in holds (re, im) pairs, coef_im the imaginary parts of the coefficients
    const int zdim = Z ? 2 : 1;
    P->cplx = Z;
    // spin-orbit plans keep U(1)_N only: every 2Sz label is 0 and the two singly occupied site states share a sector
    static const int SITE_S0[4] = {0, 0, 0, 0};
    const int* const SITE_S = Z ? SITE_S0 : dmrg::SITE_S;
    typedef std::complex<double> cplx_t;
    std::vector<cplx_t> site_z((size_t)nsite * 16);
    for (size_t i = 0; i < site_z.size(); i++) site_z[i] = Z ? cplx_t(site_ops_in[2 * i], site_ops_in[2 * i + 1]) : cplx_t(site_ops_in[i], 0.0);
    const cplx_t* site_ops = site_z.data();
    if (Z) {
        for (int side = 0; side < 2; side++)
            for (auto& sc : P->ops->sec[side]) DMRG_REQUIRE(sc.two_sz == 0, "dmrg_plan_create_z: sector labels must have two_sz = 0 (only N is a symmetry)");
        DMRG_REQUIRE(two_sz_total == 0, "dmrg_plan_create_z: two_sz_total must be 0");
    }
    int64_t nterms = nterms_in;   // shrinks to this rank's share when the plan is a shard
    const int64_t workspace_bytes = pol.workspace_bytes;
    const int64_t kMaxMergedCols = pol.max_merged_cols;
    const double kSplitWaves = pol.split_waves, kMinSplitStages = pol.min_split_stages;
    const bool kTileOrder = pol.tile_order;
    const int kSplitSmall = pol.split_small;
    P->copy_mode = pol.copy_mode;
    P->shard_rank = pol.shard_rank;
    P->shard_count = pol.shard_count;
    const bool kReleaseR = pol.release_r_store;
    DMRG_REQUIRE(!P->ops->r_released, "dmrg_plan_create: the R-side blocks of this store were released to an earlier plan (release_r_store)");
    const dmrg_ops* S = P->ops;
    const auto& secL = S->sec[0];
    const auto& secR = S->sec[1];
    const int nL = (int)secL.size(), nR = (int)secR.size();
    const int nops = (int)S->ops.size();

    // ---- psi block table, sorted by (iR, c1, c2, iL) -- each block dense row-major dL x dR --------
    std::vector<int32_t> lut((size_t)nL * 16 * nR, -1);
    {
        int64_t off = 0;
        for (int iR = 0; iR < nR; iR++)
            for (int c1 = 0; c1 < 4; c1++)
                for (int c2 = 0; c2 < 4; c2++) {
                    const int NL = n_total - secR[iR].n - SITE_N[c1] - SITE_N[c2];
                    const int SL = two_sz_total - secR[iR].two_sz - SITE_S[c1] - SITE_S[c2];
                    for (int iL = 0; iL < nL; iL++)
                        if (secL[iL].n == NL && secL[iL].two_sz == SL) {
                            lut[(((size_t)iL * 4 + c1) * 4 + c2) * nR + iR] = (int32_t)P->blocks.size();
                            P->blocks.push_back({iL, c1, c2, iR, secL[iL].dim, secR[iR].dim, off});
                            off += (int64_t)secL[iL].dim * secR[iR].dim;
                            break;
                        }
                }
        P->psi_size = off * zdim;   // doubles; block offsets count numbers (complex ones for a complex plan)
    }
    const int64_t nblk = (int64_t)P->blocks.size();
    DMRG_REQUIRE(nblk > 0, "dmrg_plan_create: no psi block has the target quantum numbers (%d, %d)", n_total, two_sz_total);

    // ---- per-op inverse sector map: rowof[op][c] = row sector r with colsec[r] == c ----------------
    std::vector<std::vector<int32_t>> rowof(nops);
    for (int o = 0; o < nops; o++) {
        const int ns = (int)S->colsec[o].size();
        rowof[o].assign(ns, -1);
        for (int r = 0; r < ns; r++)
            if (S->colsec[o][r] >= 0) rowof[o][S->colsec[o][r]] = r;
    }

    // ---- validate terms, order them so that terms sharing an R operator are adjacent ------------
    for (int64_t t = 0; t < nterms; t++) {
        const dmrg_term& T = terms[t];
        DMRG_REQUIRE(T.op_l >= -1 && T.op_l < nops && T.op_r >= -1 && T.op_r < nops, "dmrg_plan_create: term %lld: operator id out of range", (long long)t);
        DMRG_REQUIRE(T.op_l < 0 || S->ops[T.op_l].side == 0, "dmrg_plan_create: term %lld: op_l is not a left-block operator", (long long)t);
        DMRG_REQUIRE(T.op_r < 0 || S->ops[T.op_r].side == 1, "dmrg_plan_create: term %lld: op_r is not a right-block operator", (long long)t);
        DMRG_REQUIRE(T.dot1 >= 0 && T.dot1 < nsite && T.dot2 >= 0 && T.dot2 < nsite, "dmrg_plan_create: term %lld: site operator id out of range", (long long)t);
        int dn = 0, ds = 0;
        if (T.op_l >= 0) { const int s = T.trans_l ? -1 : 1; dn += s * S->ops[T.op_l].dn; ds += s * S->ops[T.op_l].d2sz; }
        if (T.op_r >= 0) { const int s = T.trans_r ? -1 : 1; dn += s * S->ops[T.op_r].dn; ds += s * S->ops[T.op_r].d2sz; }
        const cplx_t* o1 = site_ops + 16 * (size_t)T.dot1;
        const cplx_t* o2 = site_ops + 16 * (size_t)T.dot2;
        for (int a = 0; a < 4; a++) for (int b = 0; b < 4; b++) {
            if (o1[4 * a + b] == 0.0) continue;
            for (int c = 0; c < 4; c++) for (int d = 0; d < 4; d++) {
                if (o2[4 * c + d] == 0.0) continue;
                const int tn = dn + SITE_N[a] - SITE_N[b] + SITE_N[c] - SITE_N[d];
                const int ts = ds + SITE_S[a] - SITE_S[b] + SITE_S[c] - SITE_S[d];
                if (tn != 0 || ts != 0) {
                    set_error("dmrg_plan_create: term %lld does not conserve (N, 2Sz): residual (%d, %d)", (long long)t, tn, ts);
                    return DMRG_ECHARGE;
                }
            }
        }
    }
    std::vector<int64_t> order(nterms);
    for (int64_t t = 0; t < nterms; t++) order[t] = t;
    std::stable_sort(order.begin(), order.end(), [&](int64_t a, int64_t b) {
        const dmrg_term &A = terms[a], &B = terms[b];
        if (A.op_r != B.op_r) return A.op_r < B.op_r;
        if ((A.trans_r != 0) != (B.trans_r != 0)) return A.trans_r == 0;
        return false;
    });

    // ---- enumerate tasks: (term, psi block, dot transition)  (Eq. 7 at the level of blocks) ------
    // Terms are independent here: contiguous slices of the ordered term list are expanded by all host threads into slice-local
    // task lists, which are then concatenated in slice order (the result does not depend on the thread count).
    std::vector<Task> tasks;
    std::vector<int64_t> term_task_begin(nterms + 1, 0);
    std::vector<double> term_flops(nterms, 0.0);
    double canon_flops = 0.0;
    const unsigned n_enum_thr = (unsigned)std::max<int64_t>(1, std::min<int64_t>({(int64_t)std::thread::hardware_concurrency(), nterms / 64 + 1, 32}));
    std::vector<std::vector<Task>> slice_tasks(n_enum_thr);
    std::vector<int64_t> term_ntasks(nterms, 0);
    auto enumerate_slice = [&](unsigned slice) {
      std::vector<Task>& tasks = slice_tasks[slice];   // shadows the merged list on purpose
      const int64_t to_lo = nterms * slice / n_enum_thr, to_hi = nterms * (slice + 1) / n_enum_thr;
      for (int64_t to = to_lo; to < to_hi; to++) {
        const dmrg_term& T = terms[order[to]];
        const size_t ntasks_before = tasks.size();
        const cplx_t* o1 = site_ops + 16 * (size_t)T.dot1;
        const cplx_t* o2 = site_ops + 16 * (size_t)T.dot2;
        const cplx_t coef(T.coef, (Z && coef_im) ? coef_im[order[to]] : 0.0);
        const int p1 = site_parity[T.dot1] & 1, p2 = site_parity[T.dot2] & 1;
        const int pR = T.op_r >= 0 ? (S->ops[T.op_r].dn & 1) : 0;
        for (int64_t b = 0; b < nblk; b++) {
            const dmrg_psi_block& B = P->blocks[b];
            int iLo = B.il, iRo = B.ir;
            int64_t l_off = -1, r_off = -1;
            if (T.op_l >= 0) {
                if (!T.trans_l) { iLo = rowof[T.op_l][B.il]; if (iLo < 0) continue; l_off = S->row_off[T.op_l][iLo]; }
                else { l_off = S->row_off[T.op_l][B.il]; iLo = S->colsec[T.op_l][B.il]; }
                if (l_off < 0 || iLo < 0) continue;
            }
            if (T.op_r >= 0) {
                if (!T.trans_r) { iRo = rowof[T.op_r][B.ir]; if (iRo < 0) continue; r_off = S->row_off[T.op_r][iRo]; }
                else { r_off = S->row_off[T.op_r][B.ir]; iRo = S->colsec[T.op_r][B.ir]; }
                if (r_off < 0 || iRo < 0) continue;
            }
            const int Nl = secL[B.il].n;
            const int zexp = p1 * Nl + p2 * (Nl + SITE_N[B.c1]) + pR * (Nl + SITE_N[B.c1] + SITE_N[B.c2]);
            const double zeta = (zexp & 1) ? -1.0 : 1.0;
            for (int c1o = 0; c1o < 4; c1o++) {
                const cplx_t v1 = o1[4 * c1o + B.c1];
                if (v1 == 0.0) continue;
                for (int c2o = 0; c2o < 4; c2o++) {
                    const cplx_t v2 = o2[4 * c2o + B.c2];
                    if (v2 == 0.0) continue;
                    const int32_t ob = lut[(((size_t)iLo * 4 + c1o) * 4 + c2o) * nR + iRo];
                    if (ob < 0) continue;
                    Task k;
                    k.term_ord = (int32_t)to; k.in_blk = (int32_t)b; k.out_blk = ob;
                    k.l_trans = T.trans_l != 0; k.r_trans = T.trans_r != 0;
                    k.dLi = B.dl; k.dRi = B.dr; k.dLo = secL[iLo].dim; k.dRo = secR[iRo].dim;
                    k.l_off = l_off; k.r_off = r_off;
                    const cplx_t alpha = coef * zeta * v1 * v2;
                    k.alpha = alpha.real();
                    k.canon = 1;
                    if (!Z || alpha.real() != 0.0 || alpha.imag() == 0.0) tasks.push_back(k);
                    if (Z && alpha.imag() != 0.0) {   // the imaginary part of the coefficient accumulates into the second buffer
                        k.canon = alpha.real() == 0.0;
                        k.alpha = alpha.imag();
                        k.out_blk = ob + (int32_t)nblk;
                        tasks.push_back(k);
                    }
                    // a complex GEMM is 4 real ones: 8 M N K (zdim^2 = 4)
                    if (r_off >= 0) term_flops[to] += 2.0 * zdim * zdim * k.dLi * k.dRi * k.dRo;
                    if (l_off >= 0) term_flops[to] += 2.0 * zdim * zdim * k.dLo * k.dLi * k.dRo;
                }
            }
        }
        term_ntasks[to] = (int64_t)(tasks.size() - ntasks_before);
      }
    };
    {
        std::vector<std::thread> pool;
        for (unsigned t = 1; t < n_enum_thr; t++) pool.emplace_back(enumerate_slice, t);
        enumerate_slice(0);
        for (auto& th : pool) th.join();
    }
    for (int64_t to = 0; to < nterms; to++) term_task_begin[to + 1] = term_task_begin[to] + term_ntasks[to];
    tasks.reserve((size_t)term_task_begin[nterms]);
    for (auto& v : slice_tasks) { tasks.insert(tasks.end(), v.begin(), v.end()); std::vector<Task>().swap(v); }
    // ---- operator parallelism: this plan keeps one contiguous range of the ORDERED term list -----------
    // The terms are ordered by R operator, so a range needs only its own complementary operators; ranges are cut where
    // the running canonical cost crosses k/shard_count of the total.  Every rank computes the same cuts (no communication);
    // sigma = sum over ranks of the partial sigmas (one all-reduce of |psi| doubles per H psi, done by the caller).
    if (pol.shard_count > 1) {
        std::vector<double> prefix(nterms + 1, 0.0);
        for (int64_t to = 0; to < nterms; to++) prefix[to + 1] = prefix[to] + term_flops[to];
        auto cut = [&](int r) -> int64_t {
            if (r <= 0) return 0;
            if (r >= pol.shard_count) return nterms;
            const double target = prefix[nterms] * r / pol.shard_count;
            return (int64_t)(std::lower_bound(prefix.begin(), prefix.end(), target) - prefix.begin());
        };
        const int64_t lo = std::min(cut(pol.shard_rank), nterms), hi = std::max(lo, std::min(cut(pol.shard_rank + 1), nterms));
        const int64_t tb = term_task_begin[lo], te = term_task_begin[hi];
        std::vector<Task> kept(tasks.begin() + tb, tasks.begin() + te);
        for (Task& k : kept) k.term_ord -= (int32_t)lo;
        tasks.swap(kept);
        std::vector<int64_t> ttb(hi - lo + 1);
        for (int64_t to = lo; to <= hi; to++) ttb[to - lo] = term_task_begin[to] - tb;
        term_task_begin.swap(ttb);
        P->shard_terms.assign(order.begin() + lo, order.begin() + hi);
        term_flops = std::vector<double>(term_flops.begin() + lo, term_flops.begin() + hi);
        nterms = hi - lo;
    } else {
        P->shard_terms.assign(order.begin(), order.end());
    }
    for (double f : term_flops) canon_flops += f;
    P->stats[ST_TASKS] = (double)std::count_if(tasks.begin(), tasks.end(), [](const Task& k) { return k.canon != 0; });   // a complex task's imaginary-coefficient twin is not a task of its own
    P->stats[ST_CANON_FLOPS] = canon_flops;

    // ---- chunk the (ordered) terms by X workspace --------------------------------------------------
    auto x_elems = [zdim](const Task& k) { return (int64_t)k.dLi * zdim * round_up2(k.dRo); };
    int64_t ws_elems = workspace_bytes / 8;
    {   // the workspace must hold the X products of the largest single term (terms are independent here: all host threads)
        std::vector<int64_t> slice_max(n_enum_thr, 0);
        auto max_slice = [&](unsigned slice) {
            std::unordered_map<int64_t, char> seen;
            const int64_t to_lo = nterms * slice / n_enum_thr, to_hi = nterms * (slice + 1) / n_enum_thr;
            for (int64_t to = to_lo; to < to_hi; to++) {
                seen.clear();
                int64_t need = 0;
                for (int64_t i = term_task_begin[to]; i < term_task_begin[to + 1]; i++) {
                    const Task& k = tasks[i];
                    if (k.r_off < 0) continue;
                    if (seen.emplace(xkey(k.r_off, k.r_trans, k.in_blk, nblk), 1).second) need += x_elems(k);
                }
                slice_max[slice] = std::max(slice_max[slice], need);
            }
        };
        std::vector<std::thread> pool;
        for (unsigned t = 1; t < n_enum_thr; t++) pool.emplace_back(max_slice, t);
        max_slice(0);
        for (auto& th : pool) th.join();
        const int64_t max_term = *std::max_element(slice_max.begin(), slice_max.end());
        ws_elems = std::max<int64_t>(std::max(ws_elems, max_term), 2);
    }
    std::vector<int64_t> chunk_begin;   // term_ord of the first term of each chunk
    {
        std::unordered_map<int64_t, char> seen;
        int64_t used = 0;
        chunk_begin.push_back(0);
        for (int64_t to = 0; to < nterms; to++) {
            int64_t add = 0;
            std::vector<int64_t> newkeys;
            for (int64_t i = term_task_begin[to]; i < term_task_begin[to + 1]; i++) {
                const Task& k = tasks[i];
                if (k.r_off < 0) continue;
                const int64_t key = xkey(k.r_off, k.r_trans, k.in_blk, nblk);
                if (seen.emplace(key, 1).second) { add += x_elems(k); newkeys.push_back(key); }
            }
            if (used + add > ws_elems && to > chunk_begin.back()) {
                chunk_begin.push_back(to);
                seen.clear();
                used = 0;
                add = 0;
                for (int64_t i = term_task_begin[to]; i < term_task_begin[to + 1]; i++) {
                    const Task& k = tasks[i];
                    if (k.r_off < 0) continue;
                    if (seen.emplace(xkey(k.r_off, k.r_trans, k.in_blk, nblk), 1).second) add += x_elems(k);
                }
            }
            used += add;
        }
    }
    const int64_t nchunks = nterms > 0 ? (int64_t)chunk_begin.size() : 0;
    chunk_begin.push_back(nterms);
    P->stats[ST_CHUNKS] = (double)nchunks;

    // ---- build jobs / segments / tiles chunk by chunk ---------------------------------------------
    // The GEMM kernels read psi from a padded copy (rows padded to an even length, refreshed at the start of every
    // dmrg_sigma): every psi operand is then 16-byte aligned; consecutive blocks of a panel stay contiguous.
    std::vector<int64_t> ppad(nblk);
    {
        int64_t o = 0;
        for (int64_t b = 0; b < nblk; b++) { ppad[b] = o; o += (int64_t)P->blocks[b].dl * zdim * round_up2(P->blocks[b].dr); }
        P->psi_pad_elems = std::max<int64_t>(o, 2);
    }
    // psi panels (all blocks of one R sector, contiguous in the padded copy): the matrices of the stage-1 A tensor maps
    std::vector<int64_t> panel_first(nR, -1), panel_rows(nR, 0);
    for (int64_t b = 0; b < nblk; b++) {
        const int ir = P->blocks[b].ir;
        if (panel_first[ir] < 0) panel_first[ir] = b;
        panel_rows[ir] += P->blocks[b].dl;
    }
    const int TILE = kVariants[0].bm;   // square tiles: the same box rules serve A and B operands

    // The chunks are planned independently of each other by all host threads, each into its own ChunkOut with
    // chunk-local job / segment / tensor-map indices and pack offsets; they are then appended in chunk order (the
    // result does not depend on the thread count).
    struct TileList { std::vector<Tile> tiles; size_t nbig = 0, ntiles = 0; double frag_area = 0, cost = 0; };   // ntiles: BM x BN tiles (a run of M sub-tiles counts each)   // frag_area: 8x8 fragments of the tiles x 64   // sorted tiles of one stage; [0, nbig) = large-block jobs (split_small)
    struct ChunkOut {
        std::vector<Job> jobs;
        std::vector<Seg> segs;
        TileList t1, t2;
        std::vector<RedJob> reds;
        std::vector<PackDesc> packs;
        std::vector<size_t> pack_segs;
        std::vector<std::pair<int32_t, HdItem>> hd;
        MapTable maps;
        int64_t pack_top = 0, ws_peak = 0, s1_jobs = 0;
        double alg_flops = 0, s1_flops = 0, s2_flops = 0, padded_flops = 0, alg_bytes = 0, stage_flops = 0, tile_flops = 0, warp_flops = 0;
        int rc = DMRG_OK;
        std::string err;
    };
    // longest first (LPT through the hardware block scheduler); inside a sqrt(2)-wide cost bucket, stage-2
    // tiles follow `key` = (L sector of the sigma block, split-K part): sigma blocks of one L-sector row walk
    // the same L operator blocks, so launching them together lets them share those blocks in L2
    auto sort_tiles = [&](std::vector<TileRec>& r, const std::vector<Job>& jobs, const std::vector<Seg>& segs, TileList& out) {
        if (kTileOrder) {
            for (auto& x : r) x.bucket = (int32_t)std::floor(2.0 * std::log2(x.cost));
            std::stable_sort(r.begin(), r.end(), [](const TileRec& a, const TileRec& b) {
                if (a.bucket != b.bucket) return a.bucket > b.bucket;
                return a.key < b.key;
            });
        } else {
            std::stable_sort(r.begin(), r.end(), [](const TileRec& a, const TileRec& b) { return a.cost > b.cost; });
        }
        // measurement aid: tiles of small-block jobs (min(M, N, K) < split_small) move, in order, to the end of the
        // list and get a launch of their own, so that ncu reports the small-block batch (HBM-side) apart from the
        // large-block one (FP64-pipe bound).  Same kernel, same tiles, same results; default off.
        size_t nbig = r.size();
        if (kSplitSmall > 0)
            nbig = std::stable_partition(r.begin(), r.end(), [&](const TileRec& a) {
                       const Job& j = jobs[a.t.job];
                       int d = std::min(j.M, j.N);
                       if (j.seg_end - j.seg_begin == 1) d = std::min(d, segs[j.seg_begin].K);   // stage 1: K = d_R
                       return d >= kSplitSmall;
                   }) - r.begin();
        out.nbig = nbig;
        out.tiles.reserve(r.size());
        for (auto& x : r) {
            out.tiles.push_back(x.t);
            out.frag_area += frag_area(x.t.rows, x.t.cols) + (x.t.reps - 1) * frag_area(TILE, x.t.cols);
            out.ntiles += x.t.reps;
            out.cost += x.cost;
        }
    };

    auto build_chunk = [&](int64_t ch, ChunkOut& O) -> int {
        auto& jobs = O.jobs;
        auto& segs = O.segs;
        auto& reds = O.reds;
        auto& packs = O.packs;
        auto& pack_segs = O.pack_segs;
        auto& maps = O.maps;
        int64_t& pack_top = O.pack_top;
        int64_t& ws_peak = O.ws_peak;
        int64_t& s1_jobs = O.s1_jobs;
        double &alg_flops = O.alg_flops, &s1_flops = O.s1_flops, &s2_flops = O.s2_flops, &padded_flops = O.padded_flops, &alg_bytes = O.alg_bytes,
               &stage_flops = O.stage_flops, &tile_flops = O.tile_flops, &warp_flops = O.warp_flops;
        const int64_t t0 = term_task_begin[chunk_begin[ch]], t1 = term_task_begin[chunk_begin[ch + 1]];
        if (t0 == t1) return DMRG_OK;
        // -- stage 1: unique (R block, trans, psi block) products, merged into runs of consecutive psi blocks
        struct XReq { int64_t r_off; int32_t r_trans, in_blk, dRo; };
        std::vector<XReq> req;
        {
            std::unordered_map<int64_t, char> seen;
            for (int64_t i = t0; i < t1; i++) {
                const Task& k = tasks[i];
                if (k.r_off < 0) continue;
                if (seen.emplace(xkey(k.r_off, k.r_trans, k.in_blk, nblk), 1).second) req.push_back({k.r_off, k.r_trans, k.in_blk, k.dRo});
            }
        }
        std::sort(req.begin(), req.end(), [](const XReq& a, const XReq& b) {
            if (a.r_off != b.r_off) return a.r_off < b.r_off;
            if (a.r_trans != b.r_trans) return a.r_trans < b.r_trans;
            return a.in_blk < b.in_blk;
        });
        std::unordered_map<int64_t, XLoc> xloc;
        xloc.reserve(req.size() * 2);
        std::unordered_map<int64_t, std::pair<int64_t, int64_t>> pack_loc;   // (R block, trans) -> chunk-local offset of its packed copy (+ distance to its imaginary-part rows)
        std::vector<TileRec> recs1[NUM_VARIANTS];
        std::vector<std::pair<int, int>> cut_m, cut_n;
        int64_t xtop = 0;
        // runs: one R block (normal or transposed use) applied to a run of consecutive psi blocks of its input panel
        struct Run { size_t i, j; int64_t rows; };
        std::vector<Run> runs;
        for (size_t i = 0; i < req.size();) {
            size_t j = i + 1;
            while (j < req.size() && req[j].r_off == req[i].r_off && req[j].r_trans == req[i].r_trans &&
                   req[j].in_blk == req[j - 1].in_blk + 1 && P->blocks[req[j].in_blk].ir == P->blocks[req[i].in_blk].ir)
                j++;
            int64_t rows = 0;
            for (size_t q = i; q < j; q++) rows += P->blocks[req[q].in_blk].dl;
            DMRG_REQUIRE(rows < (int64_t(1) << 31), "dmrg_plan_create: merged stage-1 panel too tall");
            runs.push_back({i, j, rows});
            i = j;
        }
        // N-merge: R blocks that are applied to exactly the same runs of psi rows (same "signature") are stacked
        // along N in the plan's packed store, K-contiguous, each block once per chunk (h.c. uses transposed while
        // packing).  Every run of the signature is then ONE GEMM against the whole stack: one pass over those psi
        // rows serves hundreds of R blocks, tiles are full but for one remainder per stack, and sectors of dimension
        // 1..32 stop being skinny GEMMs.
        // `runs` is ordered by (R block, first psi block): the runs of one R block are consecutive.
        struct RBlk { size_t r0, r1; };   // range in runs[]
        std::vector<RBlk> rblks;
        for (size_t r = 0; r < runs.size();) {
            size_t e = r + 1;
            while (e < runs.size() && req[runs[e].i].r_off == req[runs[r].i].r_off && req[runs[e].i].r_trans == req[runs[r].i].r_trans) e++;
            rblks.push_back({r, e});
            r = e;
        }
        auto sig_less = [&](const RBlk& x, const RBlk& y) {   // lexicographic on the list of (first block, length)
            const size_t nx = x.r1 - x.r0, ny = y.r1 - y.r0;
            for (size_t t = 0; t < std::min(nx, ny); t++) {
                const Run &a = runs[x.r0 + t], &b = runs[y.r0 + t];
                if (req[a.i].in_blk != req[b.i].in_blk) return req[a.i].in_blk < req[b.i].in_blk;
                if (a.j - a.i != b.j - b.i) return (a.j - a.i) < (b.j - b.i);
            }
            return nx < ny;
        };
        std::stable_sort(rblks.begin(), rblks.end(), sig_less);
        for (size_t c0 = 0; c0 < rblks.size();) {
            // class [c0, c1): same signature, stack width capped
            const dmrg_psi_block& B0 = P->blocks[req[runs[rblks[c0].r0].i].in_blk];
            // complex plans: K runs over both halves of a row-planar psi row (the pad column between them meets a zero of
            // the pack), a stack holds the real-part rows of all its blocks, then their imaginary-part rows
            const int dRi = B0.dr, ldp = zdim * (int)round_up2(dRi), Keff = Z ? ldp : dRi;
            size_t c1 = c0;
            int64_t ncols = 0;
            while (c1 < rblks.size() && !sig_less(rblks[c0], rblks[c1]) && !sig_less(rblks[c1], rblks[c0]) &&
                   (c1 == c0 || ncols + zdim * round_up2(req[runs[rblks[c1].r0].i].dRo) <= kMaxMergedCols)) {
                ncols += zdim * round_up2(req[runs[rblks[c1].r0].i].dRo);
                c1++;
            }
            const int ldx = (int)ncols;   // even by construction
            const int64_t half = ncols / 2;   // complex: column (= packed row) distance between the two parts of a block
            // pack the stack once
            std::vector<int64_t> col0s;
            int64_t col0 = 0;
            for (size_t c = c0; c < c1; c++) {
                const XReq& r0 = req[runs[rblks[c].r0].i];
                packs.push_back({r0.r_off, pack_top + col0 * ldp, r0.dRo, dRi, zdim * (int32_t)round_up2(r0.r_trans ? r0.dRo : dRi), r0.r_trans, ldp, 0,
                                 Z ? half * ldp : 0});
                pack_loc[r0.r_off * 2 + r0.r_trans] = {pack_top + col0 * ldp, Z ? half * ldp : 0};
                col0s.push_back(col0);
                col0 += round_up2(r0.dRo);
                alg_bytes += 8.0 * zdim * (double)dRi * r0.dRo;
            }
            // one GEMM per run of the signature
            const size_t nruns = rblks[c0].r1 - rblks[c0].r0;
            for (size_t t = 0; t < nruns; t++) {
                const Run& R0 = runs[rblks[c0].r0 + t];
                const dmrg_psi_block& Bt = P->blocks[req[R0.i].in_blk];
                const int64_t rows = R0.rows;
                for (size_t c = c0; c < c1; c++) {
                    const Run& Rc = runs[rblks[c].r0 + t];
                    int64_t rr = 0;
                    for (size_t q = Rc.i; q < Rc.j; q++) {
                        // complex: recorded with half the row pitch -- the row-planar slice as stage 2 reads it (2 dL rows)
                        xloc[xkey(req[q].r_off, req[q].r_trans, req[q].in_blk, nblk)] = {xtop + rr * ldx + col0s[c - c0], ldx / zdim};
                        rr += P->blocks[req[q].in_blk].dl;
                    }
                    s1_flops += 2.0 * zdim * zdim * rows * dRi * req[Rc.i].dRo;
                    alg_bytes += 8.0 * zdim * rows * req[Rc.i].dRo;
                }
                alg_bytes += 8.0 * zdim * rows * dRi;
                Seg s;
                s.a_off = ppad[req[R0.i].in_blk]; s.lda = ldp;
                s.b_off = kPackBase + pack_top; s.ldb = ldp;   // resolved to an offset from the operator store at upload
                s.K = Keff; s.alpha = 1.0;
                s.flags = (SP_PSI << SEG_A_SPACE_SHIFT) | (SP_OPS << SEG_B_SPACE_SHIFT) | SEG_B_KCONTIG;
                {
                    const int64_t pf = panel_first[Bt.ir];
                    const BoxShape ba = box_shape(0, Keff, panel_rows[Bt.ir], TILE), bb = box_shape(0, Keff, ncols, TILE);
                    s.a_map = maps.get(MS_PSI, ppad[pf], 0, Keff, panel_rows[Bt.ir], ldp, ba);
                    s.a_o0 = (int32_t)((ppad[req[R0.i].in_blk] - ppad[pf]) / ldp);
                    s.b_map = maps.get(MS_PACK, pack_top, 0, Keff, ncols, ldp, bb);
                    s.a_pitch = (uint16_t)ba.inner; s.b_pitch = (uint16_t)bb.inner;
                    s.a_bytes = 8u * ba.inner * ba.outer; s.b_bytes = 8u * bb.inner * bb.outer;
                }
                pack_segs.push_back(segs.size());
                Job jb;
                jb.c_off = xtop; jb.ldc = ldx; jb.M = (int)rows; jb.N = (int)ncols;
                jb.seg_begin = (int32_t)segs.size(); jb.seg_end = jb.seg_begin + 1;
                jb.flags = (SP_X << JOB_C_SPACE_SHIFT);
                jb.nstages = (Keff + GEMM_BK - 1) / GEMM_BK;
                segs.push_back(s);
                const int v = choose_variant(jb.M, jb.N);
                const int bm = kVariants[v].bm, bn = kVariants[v].bn;
                const double kpad4 = 4.0 * ((Keff + 3) / 4);
                cut_dim(jb.M, bm, cut_m);
                cut_dim(jb.N, bn, cut_n);
                // short tiles (K = d_R is a few stages) are handed out in runs of consecutive M tiles: one CTA, one descriptor
                // fetch, the stage ring running on from tile to tile
                const size_t run = (size_t)std::min(8, std::max(1, (pol.tile_run_stages + jb.nstages - 1) / jb.nstages));
                for (size_t a0 = 0; a0 < cut_m.size(); a0 += run) {
                    const size_t a1 = std::min(cut_m.size(), a0 + run);
                    for (auto& b : cut_n) {
                        Tile t{(int32_t)jobs.size(), cut_m[a0].first, b.first, (uint16_t)cut_m[a1 - 1].second, (uint16_t)b.second};
                        t.reps = (uint16_t)(a1 - a0);
                        recs1[v].push_back({t, kpad4 * (double)(a1 - a0)});
                    }
                }
                padded_flops += 2.0 * frag_area(jb.M, jb.N) * kpad4;
                stage_flops += 2.0 * frag_area(jb.M, jb.N) * (double)GEMM_BK * jb.nstages;
                warp_flops += 2.0 * warp_area(cut_m, cut_n, v) * (double)GEMM_BK * jb.nstages;
                tile_flops += 2.0 * (double)cut_m.size() * cut_n.size() * bm * bn * (double)GEMM_BK * jb.nstages;
                jobs.push_back(jb);
                s1_jobs++;
                xtop += rows * ldx;
            }
            pack_top += ncols * ldp;
            c0 = c1;
        }
        ws_peak = std::max(ws_peak, xtop);
        sort_tiles(recs1[0], jobs, segs, O.t1);

        // -- stage 2: per sigma block, the ordered list of contributions -----------------------------
        std::vector<int64_t> idx(t1 - t0);
        for (int64_t i = 0; i < t1 - t0; i++) idx[i] = t0 + i;
        std::stable_sort(idx.begin(), idx.end(), [&](int64_t a, int64_t b) { return tasks[a].out_blk < tasks[b].out_blk; });
        // pass A: size every sigma-block job to choose the split-K granularity of this chunk
        struct Group { size_t i, j; int variant, ntm, ntn, nst; };
        std::vector<Group> groups;
        double tile_stages = 0.0;
        for (size_t i = 0; i < idx.size();) {
            size_t j = i;
            const int ob = tasks[idx[i]].out_blk;
            int nst = 0;
            while (j < idx.size() && tasks[idx[j]].out_blk == ob) {
                if (tasks[idx[j]].l_off >= 0) nst += (zdim * tasks[idx[j]].dLi + GEMM_BK - 1) / GEMM_BK;
                j++;
            }
            const dmrg_psi_block& OB = P->blocks[ob % nblk];   // complex plans: ob >= nblk = the imaginary-coefficient accumulator
            const int v = choose_variant(zdim * OB.dl, OB.dr);
            const int bm = kVariants[v].bm, bn = kVariants[v].bn;
            Group g{i, j, v, (zdim * OB.dl + bm - 1) / bm, (OB.dr + bn - 1) / bn, nst};
            // cost in units of 64x64x16 tile-stages
            tile_stages += (double)g.ntm * g.ntn * nst * (bm * bn / 4096.0);
            groups.push_back(g);
            i = j;
        }
        // A tile's K-loop is the critical path of the launch: cap it at 1/kSplitWaves of the time the whole launch
        // would take on a perfectly balanced machine, but never below kMinSplitStages.  Measured at cfg 5 (stage-2
        // ms): waves 2: 1622, 6: 1495, 24: 1375, 96: 1324, 200: 1314; floor 64 stages: 1333, 32: 1387, 16: 1409 --
        // many short parts balance better and drift apart less than few long ones; the partial tiles they
        // write (8 bytes per 2*K flops) cost nothing.
        const double smax = std::max<double>(kMinSplitStages, tile_stages / (kCtaSlots * kSplitWaves));
        std::vector<TileRec> recs2[NUM_VARIANTS];
        int64_t ptop = xtop;   // split-K partial tiles live behind the X intermediates
        std::vector<Seg> ident_segs, gemm_segs;
        for (const Group& g : groups) {
            const int ob = tasks[idx[g.i]].out_blk;
            const dmrg_psi_block& OB = P->blocks[ob % nblk];
            const int Mo = zdim * OB.dl;   // rows of the sigma block as the GEMM sees it (complex: (re, im) row pairs)
            ident_segs.clear();
            gemm_segs.clear();
            double kp4 = 0;
            for (size_t q = g.i; q < g.j; q++) {
                const Task& k = tasks[idx[q]];
                const bool ident = k.l_off < 0;
                Seg s;
                const int Ki = zdim * k.dLi, Mk = zdim * k.dLo;   // K and M extents of this contribution
                s.alpha = k.alpha;
                s.K = Ki;
                s.flags = 0;
                s.a_map = s.b_map = 0; s.a_o0 = 0; s.a_pitch = s.b_pitch = 0; s.a_bytes = s.b_bytes = 0;
                auto set_a = [&](int32_t id, BoxShape b) { s.a_map = id; s.a_pitch = (uint16_t)b.inner; s.a_bytes = 8u * b.inner * b.outer; };
                auto set_b = [&](int32_t id, BoxShape b) { s.b_map = id; s.b_pitch = (uint16_t)b.inner; s.b_bytes = 8u * b.inner * b.outer; };
                if (ident) { s.a_off = 0; s.lda = 0; s.flags |= SEG_A_IDENT; }
                else {
                    s.a_off = k.l_off; s.lda = Z ? 2 * (k.l_trans ? k.dLo : k.dLi) : (int)round_up2(k.l_trans ? k.dLo : k.dLi);
                    s.flags |= (SP_OPS << SEG_A_SPACE_SHIFT) | (k.l_trans ? SEG_A_MCONTIG : 0);
                    const BoxShape ba = box_shape(k.l_trans ? 1 : 0, Ki, Mk, TILE);
                    set_a(k.l_trans ? maps.get(MS_OPS, k.l_off, 1, Mk, Ki, s.lda, ba) : maps.get(MS_OPS, k.l_off, 0, Ki, Mk, s.lda, ba), ba);
                }
                if (k.r_off < 0) {
                    const dmrg_psi_block& IB = P->blocks[k.in_blk];
                    s.b_off = ppad[k.in_blk]; s.ldb = (int)round_up2(IB.dr);
                    s.flags |= (SP_PSI << SEG_B_SPACE_SHIFT);
                    if (ident) alg_bytes += 8.0 * zdim * k.dLi * k.dRi;
                    else { const BoxShape bb = box_shape(1, Ki, IB.dr, TILE); set_b(maps.get(MS_PSI, ppad[k.in_blk], 1, IB.dr, zdim * IB.dl, s.ldb, bb), bb); }
                } else {
                    const XLoc xl = xloc.at(xkey(k.r_off, k.r_trans, k.in_blk, nblk));
                    s.b_off = xl.off; s.ldb = xl.ld;
                    s.flags |= (SP_X << SEG_B_SPACE_SHIFT);
                    if (!ident) {   // the X slice of this task as a matrix of its own: dLi rows x dRo columns, row pitch = the stage-1 job's
                        const BoxShape bb = box_shape(1, Ki, k.dRo, TILE);
                        set_b(maps.get(MS_X, xl.off, 1, k.dRo, Ki, xl.ld, bb), bb);
                    }
                    if (k.canon) alg_flops += 2.0 * zdim * zdim * k.dLi * k.dRi * k.dRo;
                }
                if (!ident) {
                    kp4 += 4.0 * ((Ki + 3) / 4);
                    s2_flops += 2.0 * Mk * Ki * k.dRo;
                    if (k.canon) alg_flops += 2.0 * Mk * Ki * k.dRo;
                    alg_bytes += 8.0 * ((double)Mk * Ki + (double)Ki * k.dRo);
                }
                (ident ? ident_segs : gemm_segs).push_back(s);
                if (k.in_blk == k.out_blk % nblk && !Z) {
                    // diagonal term: with release_r_store the R diagonal is read from the packed copy (same pitch; a
                    // transposed copy has the same diagonal), addressed like the packed segments: kPackBase + offset
                    const int64_t r_at = k.r_off < 0 ? kHdIdent : (kReleaseR ? kPackBase + pack_loc.at(k.r_off * 2 + k.r_trans).first : k.r_off);
                    O.hd.push_back({(int32_t)ob, HdItem{k.l_off < 0 ? kHdIdent : k.l_off, r_at, (int)round_up2(k.dLi), (int)round_up2(k.dRi), k.alpha, 0, 0}});
                } else if (k.in_blk == k.out_blk % nblk) {
                    // complex plan: diag += Re((ar + i ai) l r) -- this task carries ar (accumulator 0: ar Re(l r)) or ai
                    // (accumulator 1: -ai Im(l r)).  l = (re, im) at [2i][2i] and, one image row below or -- the block used
                    // conj-transposed -- one column to the right, of the L image; r always from the packed copy "as used":
                    // re at [n][n] of the real-part rows, im at [n][n] of the imaginary-part rows.
                    const auto pl = k.r_off < 0 ? std::pair<int64_t, int64_t>{0, 0} : pack_loc.at(k.r_off * 2 + k.r_trans);
                    HdItem h{k.l_off < 0 ? kHdIdent : k.l_off, k.r_off < 0 ? kHdIdent : kPackBase + pl.first, 2 * k.dLi, 2 * (int)round_up2(k.dRi), k.alpha,
                             k.l_trans ? 1 : 2 * k.dLi, pl.second};
                    h.part = ob >= nblk;
                    O.hd.push_back({(int32_t)(ob % nblk), h});
                }
            }
            cut_dim(Mo, kVariants[g.variant].bm, cut_m);
            cut_dim(OB.dr, kVariants[g.variant].bn, cut_n);
            padded_flops += 2.0 * frag_area(Mo, OB.dr) * kp4;
            stage_flops += 2.0 * frag_area(Mo, OB.dr) * (double)GEMM_BK * g.nst;
            warp_flops += 2.0 * warp_area(cut_m, cut_n, g.variant) * (double)GEMM_BK * g.nst;
            tile_flops += 2.0 * (double)g.ntm * g.ntn * kVariants[g.variant].bm * kVariants[g.variant].bn * (double)GEMM_BK * g.nst;
            alg_bytes += 16.0 * Mo * OB.dr;
            const int nsplit = (int)std::max(1.0, std::ceil(g.nst / smax));
            int part_no = 0;
            auto push_tiles = [&](std::vector<TileRec> (&recs)[NUM_VARIANTS], int job_id, double cost) {
                const int64_t key = (int64_t)OB.il * 65536 + part_no++;
                for (auto& a : cut_m)
                    for (auto& b : cut_n) recs[g.variant].push_back({{job_id, a.first, b.first, (uint16_t)a.second, (uint16_t)b.second}, cost, key});
            };
            Job jb;
            // complex plans accumulate into the plan's own buffer: two accumulators of psi_size doubles, block b of each at twice its
            // offset, row-planar without padding (2 dl rows of dr)
            const int64_t c_at = Z ? (int64_t)(ob / nblk) * P->psi_size + 2 * OB.offset : OB.offset;
            jb.c_off = c_at; jb.ldc = OB.dr; jb.M = Mo; jb.N = OB.dr;
            jb.flags = (SP_SIGMA << JOB_C_SPACE_SHIFT) | JOB_BETA1;
            if (nsplit == 1) {
                jb.seg_begin = (int32_t)segs.size();
                segs.insert(segs.end(), ident_segs.begin(), ident_segs.end());
                segs.insert(segs.end(), gemm_segs.begin(), gemm_segs.end());
                jb.seg_end = (int32_t)segs.size();
                jb.nstages = g.nst;
                push_tiles(recs2, (int32_t)jobs.size(), g.nst + 1.0);
                jobs.push_back(jb);
            } else {
                // split-K: part p accumulates a contiguous range of segments into its own partial matrix;
                // a final job adds the partials to sigma in part order (deterministic, no atomics)
                const int ldp = (int)round_up2(OB.dr);
                const int64_t psz = (int64_t)Mo * ldp;
                size_t sbeg = 0;
                int done = 0, nparts = 0;
                std::vector<int64_t> part_off;   // consecutive: part p lives at part_off[0] + p * psz
                while (sbeg < gemm_segs.size()) {
                    const double target = (double)g.nst * (nparts + 1) / nsplit;
                    size_t send = sbeg;
                    int pst = 0;
                    while (send < gemm_segs.size() && (send == sbeg || done + pst < target)) {
                        pst += (gemm_segs[send].K + GEMM_BK - 1) / GEMM_BK;
                        send++;
                    }
                    Job pj;
                    pj.c_off = ptop; pj.ldc = ldp; pj.M = Mo; pj.N = OB.dr;
                    pj.flags = (SP_X << JOB_C_SPACE_SHIFT);
                    pj.seg_begin = (int32_t)segs.size();
                    if (nparts == 0) segs.insert(segs.end(), ident_segs.begin(), ident_segs.end());   // identity-L terms ride with part 0
                    segs.insert(segs.end(), gemm_segs.begin() + sbeg, gemm_segs.begin() + send);
                    pj.seg_end = (int32_t)segs.size();
                    pj.nstages = pst;
                    push_tiles(recs2, (int32_t)jobs.size(), pst + 1.0);
                    jobs.push_back(pj);
                    part_off.push_back(ptop);
                    ptop += psz;
                    done += pst;
                    nparts++;
                    sbeg = send;
                }
                reds.push_back({c_at, part_off[0], psz, Mo, OB.dr, ldp, nparts});
            }
            DMRG_REQUIRE(segs.size() < ((size_t)1 << 31) && jobs.size() < ((size_t)1 << 31), "dmrg_plan_create: descriptor table overflow");
        }
        ws_peak = std::max(ws_peak, ptop);
        sort_tiles(recs2[0], jobs, segs, O.t2);
        return DMRG_OK;
    };

    std::vector<ChunkOut> outs((size_t)nchunks);
    {
        const unsigned nthr = (unsigned)std::max<int64_t>(1, std::min<int64_t>({(int64_t)std::thread::hardware_concurrency(), nchunks, 32}));
        std::atomic<int64_t> next{0};
        auto worker = [&]() {
            for (int64_t ch = next.fetch_add(1); ch < nchunks; ch = next.fetch_add(1)) {
                try {
                    outs[ch].rc = build_chunk(ch, outs[ch]);
                    if (outs[ch].rc != DMRG_OK) outs[ch].err = dmrg_last_error();   // set_error is thread-local
                } catch (const std::bad_alloc&) {
                    outs[ch].rc = DMRG_ENOMEM;
                    outs[ch].err = "dmrg_plan_create: out of host memory";
                } catch (const std::exception& e) {
                    outs[ch].rc = DMRG_EINVAL;
                    outs[ch].err = std::string("dmrg_plan_create: ") + e.what();
                }
            }
        };
        std::vector<std::thread> pool;
        for (unsigned t = 1; t < nthr; t++) pool.emplace_back(worker);
        worker();
        for (auto& th : pool) th.join();
    }
    // ---- append the chunks in order ----------------------------------------------------------------------------
    std::vector<Job> jobs;
    std::vector<Seg> segs;
    std::vector<Tile> tiles;
    std::vector<std::vector<HdItem>> hd(nblk);
    std::vector<RedJob> reds;   // split-K reductions (stage 3)
    std::vector<PackDesc> packs;   // packed R store (stage-1 B operands), filled on the device after upload
    std::vector<size_t> pack_segs;  // segments whose b_off is relative to the packed store
    MapTable maps;
    int64_t pack_top = 0, ws_peak = 0, s1_jobs = 0, s1_tiles = 0, s2_tiles = 0;
    double fill_acc1 = 0, fill_acc2 = 0, cost_acc1 = 0, cost_acc2 = 0;
    double alg_flops = 0, s1_flops = 0, s2_flops = 0, padded_flops = 0, alg_bytes = 0, stage_flops = 0, tile_flops = 0, warp_flops = 0;
    // pass 1 (serial, cheap): where every chunk's tables go, the global tensor-map ids, launches, packs, diagonal items
    std::vector<size_t> job_base(nchunks), seg_base(nchunks), tile_base(nchunks);
    std::vector<int64_t> pack_base(nchunks);
    std::vector<std::vector<int32_t>> map_ids(nchunks);
    size_t njobs = 0, nsegs = 0, ntile_recs = 0;
    for (int64_t ch = 0; ch < nchunks; ch++) {
        ChunkOut& O = outs[ch];
        if (O.rc != DMRG_OK) { set_error("%s", O.err.c_str()); return O.rc; }
        job_base[ch] = njobs; seg_base[ch] = nsegs; tile_base[ch] = ntile_recs; pack_base[ch] = pack_top;
        DMRG_REQUIRE(njobs + O.jobs.size() < ((size_t)1 << 31) && nsegs + O.segs.size() < ((size_t)1 << 31), "dmrg_plan_create: descriptor table overflow");
        std::vector<int32_t>& map_id = map_ids[ch];
        map_id.resize(O.maps.descs.size());
        for (size_t m = 0; m < O.maps.descs.size(); m++) {
            MapDesc d = O.maps.descs[m];
            if (d.space == MS_PACK) d.off += pack_top;
            if (d.space == MS_PACK || d.space == MS_X) {
                // unique inside the chunk already, and a packed stack or an X slice of one chunk is no operand of another:
                // appended without the (hash) look-up that 4 M of these would cost
                map_id[m] = (int32_t)maps.descs.size();
                maps.descs.push_back(d);
            } else
                map_id[m] = maps.get(d.space, d.off, d.kind, d.inner, d.outer, d.ld, BoxShape{d.box_inner, d.box_outer});
        }
        for (size_t q : O.pack_segs) pack_segs.push_back(nsegs + q);
        for (PackDesc pd : O.packs) { pd.dst += pack_top; packs.push_back(pd); }
        for (auto& h : O.hd) {
            if (h.second.r_off >= kPackBase) h.second.r_off += pack_top;
            hd[h.first].push_back(h.second);
        }
        int stage = 1;
        size_t tile_cursor = ntile_recs;   // the chunk's tiles: stage 1 then stage 2, each list in its sorted order
        for (TileList* tl : {&O.t1, &O.t2}) {
            PlanGroup grp{stage, (int)P->launches.size(), 0};
            size_t i = 0;
            const size_t n = tl->tiles.size();
            const int variant = stage == 1 ? 1 : 0;   // 1: the instantiation whose tiles may be runs of M sub-tiles (stage 1)
            (stage == 1 ? cost_acc1 : cost_acc2) += tl->cost;
            (stage == 1 ? fill_acc1 : fill_acc2) += tl->frag_area;
            auto push_range = [&](size_t lo, size_t hi) {
                while (lo < hi) {   // grid.x limit: split very long lists
                    const size_t cnt = std::min<size_t>(hi - lo, (size_t)1 << 30);
                    P->launches.push_back({variant, stage, (int64_t)(tile_cursor + lo), (int64_t)cnt});
                    lo += cnt;
                }
            };
            if (tl->nbig > 0 && tl->nbig < n) { push_range(0, tl->nbig); i = tl->nbig; }
            push_range(i, n);
            tile_cursor += n;
            (stage == 1 ? s1_tiles : s2_tiles) += (int64_t)tl->ntiles;
            grp.nlaunch = (int)P->launches.size() - grp.first_launch;
            if (grp.nlaunch > 0) P->groups.push_back(grp);
            stage++;
        }
        if (!O.reds.empty()) {
            P->groups.push_back({3, (int)reds.size(), (int)O.reds.size()});
            reds.insert(reds.end(), O.reds.begin(), O.reds.end());
        }
        njobs += O.jobs.size(); nsegs += O.segs.size(); ntile_recs = tile_cursor;
        pack_top += O.pack_top;
        ws_peak = std::max(ws_peak, O.ws_peak);
        s1_jobs += O.s1_jobs;
        alg_flops += O.alg_flops; s1_flops += O.s1_flops; s2_flops += O.s2_flops; padded_flops += O.padded_flops; alg_bytes += O.alg_bytes;
        stage_flops += O.stage_flops; tile_flops += O.tile_flops; warp_flops += O.warp_flops;
    }
    // pass 2 (all host threads): the bulk copies -- jobs, segments (global map ids, pack offsets), tiles -- chunk by chunk
    jobs.resize(njobs);
    segs.resize(nsegs);
    tiles.resize(ntile_recs);
    {
        const unsigned nthr = (unsigned)std::max<int64_t>(1, std::min<int64_t>({(int64_t)std::thread::hardware_concurrency(), nchunks, 32}));
        std::atomic<int64_t> next{0};
        auto worker = [&]() {
            for (int64_t ch = next.fetch_add(1); ch < nchunks; ch = next.fetch_add(1)) {
                ChunkOut& O = outs[ch];
                const std::vector<int32_t>& map_id = map_ids[ch];
                const size_t jb0 = job_base[ch], sg0 = seg_base[ch];
                for (size_t j = 0; j < O.jobs.size(); j++) {
                    Job jb = O.jobs[j];
                    jb.seg_begin += (int32_t)sg0; jb.seg_end += (int32_t)sg0;
                    jobs[jb0 + j] = jb;
                }
                for (size_t q = 0; q < O.segs.size(); q++) {
                    Seg sg = O.segs[q];
                    if (!(sg.flags & SEG_A_IDENT)) { sg.a_map = map_id[sg.a_map]; sg.b_map = map_id[sg.b_map]; }
                    segs[sg0 + q] = sg;
                }
                for (size_t q : O.pack_segs) segs[sg0 + q].b_off += pack_base[ch];
                size_t tpos = tile_base[ch];
                for (TileList* tl : {&O.t1, &O.t2})
                    for (Tile t : tl->tiles) { t.job += (int32_t)jb0; tiles[tpos++] = t; }
                O = ChunkOut();   // release the chunk's host memory
                std::vector<int32_t>().swap(map_ids[ch]);
            }
        };
        std::vector<std::thread> pool;
        for (unsigned t = 1; t < nthr; t++) pool.emplace_back(worker);
        worker();
        for (auto& th : pool) th.join();
    }

    P->stats[ST_ALG_FLOPS] = alg_flops;
    P->stats[ST_S1_FLOPS] = s1_flops;
    P->stats[ST_S2_FLOPS] = s2_flops;
    P->stats[ST_PADDED_FLOPS] = padded_flops;
    P->stats[ST_STAGE_FLOPS] = stage_flops;   // K padded to whole GEMM_BK-wide stages per segment
    P->stats[ST_WARP_FLOPS] = warp_flops;     // ... M, N padded to the most loaded warp of each tile
    P->stats[ST_TILE_FLOPS] = tile_flops;     // ... and M, N padded to whole tiles: what a fill-independent tile time costs
    P->stats[ST_S1_JOBS] = (double)s1_jobs;
    P->stats[ST_LAUNCHES] = (double)P->launches.size() + (double)std::count_if(P->groups.begin(), P->groups.end(), [](const PlanGroup& g) { return g.stage == 3; });
    P->stats[ST_ALG_BYTES] = alg_bytes + 8.0 * P->psi_size;
    P->stats[ST_S1_TILES] = (double)s1_tiles;
    P->stats[ST_S2_TILES] = (double)s2_tiles;

    // ---- H diagonal lists (tasks with out == in) --------------------------------------
    std::vector<HdItem> hd_items;
    std::vector<HdBlock> hd_blocks(nblk);
    for (int64_t b = 0; b < nblk; b++) {
        hd_blocks[b] = {P->blocks[b].offset, P->blocks[b].dl, P->blocks[b].dr, (int32_t)hd_items.size(), 0, ppad[b]};
        hd_items.insert(hd_items.end(), hd[b].begin(), hd[b].end());
        hd_blocks[b].item_end = (int32_t)hd_items.size();
    }
    P->n_hd_blocks = nblk;
    std::vector<HdTile> hd_tiles;
    for (int64_t b = 0; b < nblk; b++)
        for (int ti = 0; ti < (P->blocks[b].dl + 31) / 32; ti++)
            for (int tj = 0; tj < (P->blocks[b].dr + 31) / 32; tj++) hd_tiles.push_back({(int32_t)b, (int16_t)ti, (int16_t)tj});
    P->n_hd_tiles = (int64_t)hd_tiles.size();

    // ---- upload ---------------------------------------------------------------------------------------
    P->xws_elems = std::max<int64_t>(ws_peak, 2);
    P->stats[ST_XWS_ELEMS] = (double)P->xws_elems;
    P->stats[ST_TENSOR_MAPS] = (double)maps.descs.size();
    P->stats[ST_S1_FILL] = s1_tiles ? fill_acc1 / (4096.0 * s1_tiles) : 0.0;
    P->stats[ST_S2_FILL] = s2_tiles ? fill_acc2 / (4096.0 * s2_tiles) : 0.0;
    P->stats[ST_S1_STAGES] = s1_tiles ? cost_acc1 / s1_tiles : 0.0;   // stage-1 tile cost = K padded to 4
    P->stats[ST_S2_STAGES] = s2_tiles ? cost_acc2 / s2_tiles - 1.0 : 0.0;
    P->stats[ST_DEVICE_BYTES] = (double)(segs.size() * sizeof(Seg) + tiles.size() * sizeof(TileDesc) +
                                         hd_items.size() * sizeof(HdItem) + hd_blocks.size() * sizeof(HdBlock) + maps.descs.size() * sizeof(TensorMap) +
                                         8.0 * P->xws_elems + 8.0 * pack_top + 8.0 * P->psi_pad_elems + (Z ? 16.0 * P->psi_size : 0.0));
    if (S->structure_only) return DMRG_OK;
    auto up = [&](void** dptr, const void* src, size_t bytes) -> int {
        DMRG_CUDA(cudaMalloc(dptr, std::max<size_t>(bytes, 16)));
        if (bytes) DMRG_CUDA(cudaMemcpy(*dptr, src, bytes, cudaMemcpyHostToDevice));
        return DMRG_OK;
    };
    DMRG_CUDA(cudaMalloc(&P->d_psi_pad, sizeof(double) * (size_t)P->psi_pad_elems));
    if (Z) DMRG_CUDA(cudaMalloc(&P->d_sigz, sizeof(double) * (size_t)std::max<int64_t>(2 * P->psi_size, 2)));
    // release_r_store near the memory limit: the R-side originals and their packed copy do not fit side by side.  The R side
    // is then parked on the HOST, its device allocation freed before the pack is allocated, and the pack filled from
    // staging windows (below).  Chosen when the free memory does not cover pack + X workspace + tensor maps, or forced (2).
    std::vector<double> host_r;
    int64_t host_r_rel0 = 0;   // offset of the R-side allocation in the store's address space (doubles)
    if (kReleaseR && S->side_alloc[1]) {
        size_t free_b = 0, total_b = 0;
        DMRG_CUDA(cudaMemGetInfo(&free_b, &total_b));
        const double need = 8.0 * (double)pack_top + 8.0 * (double)P->xws_elems + 8.0 * (double)P->psi_pad_elems + 128.0 * (double)maps.descs.size() +
                            64.0 * (double)tiles.size() + 64.0 * (double)segs.size() + 2e9;
        if (pol.release_staged || need > (double)free_b) {
            dmrg_ops* Sm = const_cast<dmrg_ops*>(S);
            host_r_rel0 = (int64_t)(Sm->side_alloc[1] - Sm->d_values);
            host_r.resize(Sm->side_bytes[1] / sizeof(double));
            DMRG_CUDA(cudaMemcpy(host_r.data(), Sm->side_alloc[1], Sm->side_bytes[1], cudaMemcpyDeviceToHost));
            cudaFree(Sm->side_alloc[1]);
            Sm->owned.erase(std::remove(Sm->owned.begin(), Sm->owned.end(), Sm->side_alloc[1]), Sm->owned.end());
            Sm->device_bytes -= (int64_t)Sm->side_bytes[1];
            Sm->side_alloc[1] = nullptr;
            Sm->side_bytes[1] = 0;
            Sm->r_released = true;
        }
    }
    DMRG_CUDA(cudaMalloc(&P->d_pack, sizeof(double) * (size_t)std::max<int64_t>(pack_top, 2)));
    DMRG_CUDA(cudaMemset(P->d_pack, 0, sizeof(double) * (size_t)std::max<int64_t>(pack_top, 2)));
    {   // the GEMM kernel addresses the packed store relative to the operator store (one flat device address space)
        const int64_t delta = (int64_t)(P->d_pack - S->d_values);
        for (size_t q : pack_segs) segs[q].b_off += delta - kPackBase;
    }
    for (Seg& sg : segs) sg.flags |= sg.alpha == 1.0 ? SEG_ALPHA_ONE : (sg.alpha == -1.0 ? SEG_ALPHA_NEG : 0u);
    {
        const int64_t delta = (int64_t)(P->d_pack - S->d_values);
        for (HdItem& h : hd_items) if (h.r_off >= kPackBase) h.r_off += delta - kPackBase;
    }
    int rc;
    if ((rc = up((void**)&P->d_segs, segs.data(), segs.size() * sizeof(Seg)))) return rc;
    {
        const std::vector<TileDesc> td = make_tile_descs(tiles, jobs, segs);
        if ((rc = up((void**)&P->d_tiles, td.data(), td.size() * sizeof(TileDesc)))) return rc;
    }
    if ((rc = up((void**)&P->d_reds, reds.data(), reds.size() * sizeof(RedJob)))) return rc;
    if ((rc = up((void**)&P->d_hd_items, hd_items.data(), hd_items.size() * sizeof(HdItem)))) return rc;
    if ((rc = up((void**)&P->d_hd_blocks, hd_blocks.data(), hd_blocks.size() * sizeof(HdBlock)))) return rc;
    if ((rc = up((void**)&P->d_hd_tiles, hd_tiles.data(), hd_tiles.size() * sizeof(HdTile)))) return rc;
    DMRG_CUDA(cudaMalloc(&P->d_xws, sizeof(double) * (size_t)P->xws_elems));
    {   // tensor maps hold absolute device addresses: encoded once every buffer they point into exists
        double* const base[4] = {S->d_values, P->d_xws, P->d_psi_pad, P->d_pack};
        std::vector<TensorMap> tm;
        if ((rc = encode_tensor_maps(maps.descs, base, tm))) return rc;
        if ((rc = up((void**)&P->d_tmaps, tm.data(), tm.size() * sizeof(TensorMap)))) return rc;
    }
    if (!packs.empty() && !host_r.empty()) {
        // staged fill: packs in the order of their source blocks, windows of the parked R side copied back one at a time
        std::sort(packs.begin(), packs.end(), [](const PackDesc& a, const PackDesc& b) { return a.src < b.src; });
        auto extent = [](const PackDesc& d) { return (int64_t)(d.trans ? d.dRi : d.dRo) * d.src_ld; };
        int64_t win = int64_t(1) << 29;   // 4 GiB of doubles
        for (const PackDesc& d : packs) win = std::max(win, extent(d));
        win = std::min<int64_t>(win, (int64_t)host_r.size());
        double* d_stage = nullptr;
        PackDesc* d_packs = nullptr;
        DMRG_CUDA(cudaMalloc(&d_stage, sizeof(double) * (size_t)std::max<int64_t>(win, 2)));
        DMRG_CUDA(cudaMalloc(&d_packs, packs.size() * sizeof(PackDesc)));
        DMRG_CUDA(cudaMemcpy(d_packs, packs.data(), packs.size() * sizeof(PackDesc), cudaMemcpyHostToDevice));
        for (size_t i0 = 0; i0 < packs.size();) {
            const int64_t w0 = packs[i0].src;
            size_t i1 = i0;
            int64_t w1 = w0;
            while (i1 < packs.size() && packs[i1].src + extent(packs[i1]) - w0 <= win) { w1 = std::max(w1, packs[i1].src + extent(packs[i1])); i1++; }
            DMRG_REQUIRE(i1 > i0 && w0 >= host_r_rel0 && w1 - host_r_rel0 <= (int64_t)host_r.size(), "dmrg_plan_create: packed-store source outside the R side of the store");
            DMRG_CUDA(cudaMemcpy(d_stage, host_r.data() + (w0 - host_r_rel0), sizeof(double) * (size_t)(w1 - w0), cudaMemcpyHostToDevice));
            const double* ops_win = d_stage - w0;   // address arithmetic only: ops_win[src + x] = d_stage[src - w0 + x]
            for (size_t y0 = i0; y0 < i1; y0 += 32768) {
                const unsigned ny = (unsigned)std::min<size_t>(32768, i1 - y0);
                if (Z) pack_r_z_kernel<<<dim3(4, ny), 256>>>(d_packs + y0, ops_win, P->d_pack);
                else pack_r_kernel<<<dim3(4, ny), 256>>>(d_packs + y0, ops_win, P->d_pack);
            }
            DMRG_CUDA(cudaGetLastError());
            DMRG_CUDA(cudaDeviceSynchronize());
            i0 = i1;
        }
        cudaFree(d_packs);
        cudaFree(d_stage);
        std::vector<double>().swap(host_r);
    } else if (!packs.empty()) {
        PackDesc* d_packs = nullptr;
        DMRG_CUDA(cudaMalloc(&d_packs, packs.size() * sizeof(PackDesc)));
        DMRG_CUDA(cudaMemcpy(d_packs, packs.data(), packs.size() * sizeof(PackDesc), cudaMemcpyHostToDevice));
        for (size_t y0 = 0; y0 < packs.size(); y0 += 32768) {
            const unsigned ny = (unsigned)std::min<size_t>(32768, packs.size() - y0);
            if (Z) pack_r_z_kernel<<<dim3(4, ny), 256>>>(d_packs + y0, S->d_values, P->d_pack);
            else pack_r_kernel<<<dim3(4, ny), 256>>>(d_packs + y0, S->d_values, P->d_pack);
        }
        DMRG_CUDA(cudaGetLastError());
        DMRG_CUDA(cudaDeviceSynchronize());
        cudaFree(d_packs);
    }
    if (kReleaseR && S->side_alloc[1]) {
        // nothing reads the R-side originals any more (stage 1 and the diagonal use the packed copy): give the memory back
        dmrg_ops* Sm = const_cast<dmrg_ops*>(S);
        cudaFree(Sm->side_alloc[1]);
        Sm->owned.erase(std::remove(Sm->owned.begin(), Sm->owned.end(), Sm->side_alloc[1]), Sm->owned.end());
        Sm->device_bytes -= (int64_t)Sm->side_bytes[1];
        Sm->side_alloc[1] = nullptr;
        Sm->side_bytes[1] = 0;
        Sm->r_released = true;
    }
    return gemm_init();
}

// packed[n * ldp + k] = R block element (n, k) of the operator as USED: the stored block for a normal use, its
// transpose for an h.c. use.  Run once per plan.     grid (chunks of elements, blocks)
__global__ void __launch_bounds__(256) pack_r_kernel(const PackDesc* __restrict__ descs, const double* __restrict__ ops,
                                                     double* __restrict__ pack) {
    const PackDesc d = descs[blockIdx.y];
    const int64_t n_el = (int64_t)d.dRo * d.dRi;
    for (int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; e < n_el; e += (int64_t)gridDim.x * blockDim.x) {
        int n, k;
        if (d.trans) { k = (int)(e / d.dRo); n = (int)(e - (int64_t)k * d.dRo); }   // coalesced read of the stored rows
        else { n = (int)(e / d.dRi); k = (int)(e - (int64_t)n * d.dRi); }
        const double v = d.trans ? ops[d.src + (int64_t)k * d.src_ld + n] : ops[d.src + (int64_t)n * d.src_ld + k];
        pack[d.dst + (int64_t)n * d.ldp + k] = v;
    }
}

// Complex plans: the real image of the R block as used (normal, or conj-transposed for an h.c. use), K-contiguous over both
// halves of a row-planar psi row:   real-part row n = [ re R(n, :) | -im R(n, :) ],  imaginary-part row n = [ im R(n, :) | re R(n, :) ]
// (halves of ldp / 2, pads stay zero).  The store keeps R blocks row-planar (ops_store.cu, mode 2).
__global__ void __launch_bounds__(256) pack_r_z_kernel(const PackDesc* __restrict__ descs, const double* __restrict__ ops,
                                                       double* __restrict__ pack) {
    const PackDesc d = descs[blockIdx.y];
    const int64_t n_el = (int64_t)d.dRo * d.dRi;
    const int sh = d.src_ld / 2, kh = d.ldp / 2;
    for (int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; e < n_el; e += (int64_t)gridDim.x * blockDim.x) {
        int n, k;
        double re, im;
        if (d.trans) {
            k = (int)(e / d.dRo); n = (int)(e - (int64_t)k * d.dRo);
            re = ops[d.src + (int64_t)k * d.src_ld + n];
            im = -ops[d.src + (int64_t)k * d.src_ld + sh + n];
        } else {
            n = (int)(e / d.dRi); k = (int)(e - (int64_t)n * d.dRi);
            re = ops[d.src + (int64_t)n * d.src_ld + k];
            im = ops[d.src + (int64_t)n * d.src_ld + sh + k];
        }
        double* r0 = pack + d.dst + (int64_t)n * d.ldp;
        double* r1 = r0 + d.im_delta;
        r0[k] = re; r0[kh + k] = -im;
        r1[k] = im; r1[kh + k] = re;
    }
}

// complex plans: interleaved psi -> row-planar padded copy (row i of a block = [re | im], halves of round_up2(dr))
__global__ void __launch_bounds__(256) pad_psi_z_kernel(const HdBlock* __restrict__ blocks, const double* __restrict__ psi,
                                                        double* __restrict__ pad) {
    const HdBlock b = blocks[blockIdx.y];
    const int pc = (b.dr + 1) & ~1, ld = 2 * pc;
    const int64_t n = (int64_t)b.dl * ld;
    for (int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; e < n; e += (int64_t)gridDim.x * blockDim.x) {
        const int i = (int)(e / ld), jj = (int)(e - (int64_t)i * ld);
        const int part = jj >= pc, j = jj - part * pc;
        pad[b.pad_off + e] = j < b.dr ? psi[2 * (b.offset + (int64_t)i * b.dr + j) + part] : 0.0;
    }
}

// complex plans: sigma = acc0 + i acc1, row-planar accumulators (block b at twice its offset: rows 2i, 2i+1 = re, im of
// row i) -> interleaved (re, im) pairs in the caller's vector
__global__ void __launch_bounds__(256) sigma_z_finish_kernel(const HdBlock* __restrict__ blocks, const double* __restrict__ acc0,
                                                             const double* __restrict__ acc1, double* __restrict__ sigma) {
    const HdBlock b = blocks[blockIdx.y];
    const int64_t n = (int64_t)b.dl * b.dr;
    const double* a0 = acc0 + 2 * b.offset;
    const double* a1 = acc1 + 2 * b.offset;
    for (int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; e < n; e += (int64_t)gridDim.x * blockDim.x) {
        const int i = (int)(e / b.dr), j = (int)(e - (int64_t)i * b.dr);
        const int64_t pr = (int64_t)(2 * i) * b.dr + j, pi = pr + b.dr;
        sigma[2 * (b.offset + e)] = a0[pr] - a1[pi];
        sigma[2 * (b.offset + e) + 1] = a0[pi] + a1[pr];
    }
}

// complex plans: Hd[blk][i][j] = sum_items Re(alpha l_ii r_jj), written to both the real and the imaginary slot of the
// element (the Davidson preconditioner acts on the vector as 2n reals).  A task carries the real part of its coefficient
// (part 0: + ar Re(l r)) or the imaginary part (part 1: - ai Im(l r)).  One thread per element, items in plan order.
__global__ void __launch_bounds__(256) hdiag_z_kernel(const HdBlock* __restrict__ blocks, const HdTile* __restrict__ tiles,
                                                      const HdItem* __restrict__ items, const double* __restrict__ ops,
                                                      double* __restrict__ diag) {
    const HdTile t = tiles[blockIdx.x];
    const HdBlock b = blocks[t.blk];
    const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
    const int j = t.tj * 32 + tx;
    for (int u = 0; u < 4; u++) {
        const int i = t.ti * 32 + ty + 8 * u;
        if (i >= b.dl || j >= b.dr) continue;
        double acc = 0.0;
        for (int q = b.item_begin; q < b.item_end; q++) {
            const HdItem h = items[q];
            double lr = 1.0, li = 0.0, rr = 1.0, ri = 0.0;
            if (h.l_off != kHdIdent) { const double* p = ops + h.l_off + (int64_t)(2 * i) * h.ldl + 2 * i; lr = p[0]; li = p[h.l_im]; }
            if (h.r_off != kHdIdent) { const double* p = ops + h.r_off + (int64_t)j * h.ldr + j; rr = p[0]; ri = p[h.r_im]; }
            acc += h.part ? -h.alpha * (lr * ri + li * rr) : h.alpha * (lr * rr - li * ri);
        }
        diag[2 * (b.offset + (int64_t)i * b.dr + j)] = acc;
        diag[2 * (b.offset + (int64_t)i * b.dr + j) + 1] = acc;
    }
}

// padded psi copy: block rows get an even length (zero pad)     grid (chunks, blocks)
__global__ void __launch_bounds__(256) pad_psi_kernel(const HdBlock* __restrict__ blocks, const double* __restrict__ psi,
                                                      double* __restrict__ pad) {
    const HdBlock b = blocks[blockIdx.y];
    const int ld = (b.dr + 1) & ~1;
    const int64_t n = (int64_t)b.dl * ld;
    for (int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; e < n; e += (int64_t)gridDim.x * blockDim.x) {
        const int i = (int)(e / ld), j = (int)(e - (int64_t)i * ld);
        pad[b.pad_off + e] = j < b.dr ? psi[b.offset + (int64_t)i * b.dr + j] : 0.0;
    }
}

// sigma_blk += sum_p partial_p, parts added in order (the deterministic end of split-K)     grid (chunks, jobs)
__global__ void __launch_bounds__(256) splitk_reduce_kernel(const RedJob* __restrict__ reds, const double* __restrict__ xws,
                                                            double* __restrict__ sigma) {
    const RedJob r = reds[blockIdx.y];
    const int64_t n = (int64_t)r.M * r.N;
    for (int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; e < n; e += (int64_t)gridDim.x * blockDim.x) {
        const int i = (int)(e / r.N), j = (int)(e - (int64_t)i * r.N);
        const double* p = xws + r.part_off + (int64_t)i * r.ldp + j;
        double acc = sigma[r.sigma_off + e];
        for (int k = 0; k < r.nparts; k++) acc += p[(int64_t)k * r.part_stride];
        sigma[r.sigma_off + e] = acc;
    }
}

// Hd[blk][i][j] = sum_items alpha * (L ? L[i][i] : 1) * (R ? R[j][j] : 1), items in plan order.
// One CTA per 32 x 32 tile of a block: the diagonals of 32 items at a time are staged in shared memory
// (2 x 32 values per item instead of two global reads per element and item), then every thread
// accumulates its 4 elements -- a rank-(number of items) update, deterministic.
__global__ void __launch_bounds__(256) hdiag_kernel(const HdBlock* __restrict__ blocks, const HdTile* __restrict__ tiles,
                                                    const HdItem* __restrict__ items, const double* __restrict__ ops,
                                                    double* __restrict__ diag) {
    __shared__ double sl[32][33], sr[32][33], sa[32];
    const HdTile t = tiles[blockIdx.x];
    const HdBlock b = blocks[t.blk];
    const int i0 = t.ti * 32, j0 = t.tj * 32;
    const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;   // ty 0..7
    double acc[4] = {0.0, 0.0, 0.0, 0.0};
    for (int base = b.item_begin; base < b.item_end; base += 32) {
        const int nit = min(32, b.item_end - base);
        __syncthreads();
        for (int q = ty; q < nit; q += 8) {   // item q: lane tx fetches L[i0+tx][i0+tx] and R[j0+tx][j0+tx]
            const HdItem h = items[base + q];
            const int i = i0 + tx, j = j0 + tx;
            sl[q][tx] = (h.l_off != kHdIdent && i < b.dl) ? ops[h.l_off + (int64_t)i * h.ldl + i] : 1.0;
            sr[q][tx] = (h.r_off != kHdIdent && j < b.dr) ? ops[h.r_off + (int64_t)j * h.ldr + j] : 1.0;
            if (tx == 0) sa[q] = h.alpha;
        }
        __syncthreads();
        for (int q = 0; q < nit; q++) {
            const double r = sa[q] * sr[q][tx];
#pragma unroll
            for (int u = 0; u < 4; u++) acc[u] = fma(sl[q][ty + 8 * u], r, acc[u]);
        }
    }
#pragma unroll
    for (int u = 0; u < 4; u++) {
        const int i = i0 + ty + 8 * u, j = j0 + tx;
        if (i < b.dl && j < b.dr) diag[b.offset + (int64_t)i * b.dr + j] = acc[u];
    }
}

}  // namespace dmrg

using namespace dmrg;

extern "C" {

int dmrg_plan_create(const dmrg_ops* ops, const dmrg_term* terms, int64_t nterms, const double* site_ops,
                     const int32_t* site_parity, int32_t nsite, int32_t n_total, int32_t two_sz_total,
                     int64_t workspace_bytes, dmrg_plan** out) {
    dmrg_plan_options o = {};
    o.workspace_bytes = workspace_bytes;
    return dmrg_plan_create_opts(ops, terms, nterms, site_ops, site_parity, nsite, n_total, two_sz_total, &o, out);
}

static int plan_create_any(const dmrg_ops* ops, const dmrg_term* terms, const double* coef_im, int64_t nterms, const double* site_ops,
                           const int32_t* site_parity, int32_t nsite, int32_t n_total, int32_t two_sz_total,
                           const dmrg_plan_options* options, dmrg_plan** out);

int dmrg_plan_create_opts(const dmrg_ops* ops, const dmrg_term* terms, int64_t nterms, const double* site_ops,
                          const int32_t* site_parity, int32_t nsite, int32_t n_total, int32_t two_sz_total,
                          const dmrg_plan_options* options, dmrg_plan** out) {
    if (ops && ops->cplx) { set_error("dmrg_plan_create: the store is complex (dmrg_ops_load_z): use dmrg_plan_create_z"); return DMRG_EINVAL; }
    return plan_create_any(ops, terms, nullptr, nterms, site_ops, site_parity, nsite, n_total, two_sz_total, options, out);
}

int dmrg_plan_create_z(const dmrg_ops* ops, const dmrg_term* terms, const double* coef_im, int64_t nterms, const double* site_ops,
                       const int32_t* site_parity, int32_t nsite, int32_t n_total, const dmrg_plan_options* options, dmrg_plan** out) {
    if (ops && !ops->cplx) { set_error("dmrg_plan_create_z: the store is real (dmrg_ops_load): use dmrg_plan_create"); return DMRG_EINVAL; }
    return plan_create_any(ops, terms, coef_im, nterms, site_ops, site_parity, nsite, n_total, 0, options, out);
}

int32_t dmrg_plan_is_complex(const dmrg_plan* P) { return P && P->cplx ? 1 : 0; }

static int plan_create_any(const dmrg_ops* ops, const dmrg_term* terms, const double* coef_im, int64_t nterms, const double* site_ops,
                           const int32_t* site_parity, int32_t nsite, int32_t n_total, int32_t two_sz_total,
                           const dmrg_plan_options* options, dmrg_plan** out) {
    if (!out) { set_error("dmrg_plan_create: out is NULL"); return DMRG_EINVAL; }
    *out = nullptr;
    if (!ops || nterms < 0 || (nterms > 0 && !terms) || !site_ops || !site_parity || nsite <= 0) {
        set_error("dmrg_plan_create: NULL or empty argument");
        return DMRG_EINVAL;
    }
    if (options && options->shard_count > 1 && (options->shard_rank < 0 || options->shard_rank >= options->shard_count)) {
        set_error("dmrg_plan_create: shard_rank %d outside [0, %d)", options->shard_rank, options->shard_count);
        return DMRG_EINVAL;
    }
    dmrg_plan* P = new (std::nothrow) dmrg_plan();
    if (!P) { set_error("dmrg_plan_create: out of host memory"); return DMRG_ENOMEM; }
    P->ops = ops;
    int rc;
    try {
        rc = plan_build(P, terms, coef_im, nterms, site_ops, site_parity, nsite, n_total, two_sz_total, make_policy(options));
    } catch (const std::bad_alloc&) {
        set_error("dmrg_plan_create: out of host memory");
        rc = DMRG_ENOMEM;
    } catch (const std::exception& e) {
        set_error("dmrg_plan_create: %s", e.what());
        rc = DMRG_EINVAL;
    }
    if (rc != DMRG_OK) { dmrg_plan_destroy(P); return rc; }
    *out = P;
    return DMRG_OK;
}

void dmrg_plan_destroy(dmrg_plan* P) {
    if (!P) return;
    cudaFree(P->d_segs); cudaFree(P->d_tiles); cudaFree(P->d_xws);
    cudaFree(P->d_hd_items); cudaFree(P->d_hd_blocks); cudaFree(P->d_hd_tiles); cudaFree(P->d_reds); cudaFree(P->d_pack); cudaFree(P->d_psi_pad); cudaFree(P->d_host_io); cudaFree(P->d_tmaps); cudaFree(P->d_sigz);
    for (auto e : P->ev) cudaEventDestroy(e);
    if (P->dav) davidson_ws_free(P->dav);
    delete P;
}

int64_t dmrg_plan_psi_size(const dmrg_plan* P) { return P ? P->psi_size : 0; }
int64_t dmrg_plan_num_psi_blocks(const dmrg_plan* P) { return P ? (int64_t)P->blocks.size() : 0; }
int dmrg_plan_psi_layout(const dmrg_plan* P, dmrg_psi_block* out) {
    if (!P || !out) { set_error("dmrg_plan_psi_layout: NULL argument"); return DMRG_EINVAL; }
    std::copy(P->blocks.begin(), P->blocks.end(), out);
    return DMRG_OK;
}
int64_t dmrg_plan_shard_terms(const dmrg_plan* P, int64_t* out, int64_t capacity) {
    if (!P) return 0;
    const int64_t n = (int64_t)P->shard_terms.size();
    if (out) std::copy(P->shard_terms.begin(), P->shard_terms.begin() + std::min(n, capacity), out);
    return n;
}
double dmrg_plan_stat(const dmrg_plan* P, int32_t key) { return (P && key >= 0 && key < ST_COUNT) ? P->stats[key] : -1.0; }

int dmrg_plan_set_timing(dmrg_plan* P, int32_t enable) {
    if (!P) { set_error("dmrg_plan_set_timing: NULL plan"); return DMRG_EINVAL; }
    if (enable && P->ev.empty()) {
        P->ev.resize(2 * P->groups.size() + 2);
        for (auto& e : P->ev) DMRG_CUDA(cudaEventCreate(&e));
    }
    P->timing = enable != 0;
    P->timing_valid = false;
    return DMRG_OK;
}

double dmrg_plan_stage_ms(dmrg_plan* P, int32_t which) {
    if (!P || !P->timing_valid) { set_error("dmrg_plan_stage_ms: no timed dmrg_sigma call"); return -1.0; }
    const size_t ng = P->groups.size();
    if (cudaEventSynchronize(P->ev[2 * ng + 1]) != cudaSuccess) { set_error("dmrg_plan_stage_ms: event sync failed"); return -1.0; }
    float ms = 0.f;
    if (which == 2) { cudaEventElapsedTime(&ms, P->ev[2 * ng], P->ev[2 * ng + 1]); return ms; }
    double tot = 0.0;
    for (size_t i = 0; i < ng; i++)
        if ((which == 0 && P->groups[i].stage == 1) || (which == 1 && P->groups[i].stage >= 2)) {
            cudaEventElapsedTime(&ms, P->ev[2 * i], P->ev[2 * i + 1]);
            tot += ms;
        }
    return tot;
}

int dmrg_sigma(dmrg_plan* P, const double* psi, double* sigma, void* cuda_stream) {
    if (!P || !psi || !sigma) { set_error("dmrg_sigma: NULL argument"); return DMRG_EINVAL; }
    if (((uintptr_t)psi & 15) || ((uintptr_t)sigma & 15)) { set_error("dmrg_sigma: psi and sigma must be 16-byte aligned"); return DMRG_EINVAL; }
    if (psi == sigma) { set_error("dmrg_sigma: psi and sigma must not alias"); return DMRG_EINVAL; }
    if (P->ops->structure_only) { set_error("dmrg_sigma: the operator store was loaded without values (planning only)"); return DMRG_EINVAL; }
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const size_t ng = P->groups.size();
    if (P->timing) DMRG_CUDA(cudaEventRecord(P->ev[2 * ng], st));
    // complex plans accumulate in their own row-planar buffers (two accumulators) and write sigma out at the end
    double* const acc = P->cplx ? P->d_sigz : sigma;
    DMRG_CUDA(cudaMemsetAsync(acc, 0, sizeof(double) * (size_t)P->psi_size * (P->cplx ? 2 : 1), st));
    for (int64_t y0 = 0; y0 < P->n_hd_blocks; y0 += 32768) {
        const unsigned ny = (unsigned)std::min<int64_t>(32768, P->n_hd_blocks - y0);
        if (P->cplx) pad_psi_z_kernel<<<dim3(8, ny), 256, 0, st>>>(P->d_hd_blocks + y0, psi, P->d_psi_pad);
        else pad_psi_kernel<<<dim3(8, ny), 256, 0, st>>>(P->d_hd_blocks + y0, psi, P->d_psi_pad);
    }
    DMRG_CUDA(cudaGetLastError());
    for (size_t gi = 0; gi < ng; gi++) {
        const PlanGroup& G = P->groups[gi];
        if (P->timing) DMRG_CUDA(cudaEventRecord(P->ev[2 * gi], st));
        if (G.stage == 3) {   // first_launch / nlaunch index the reduction table here
            for (int y0 = 0; y0 < G.nlaunch; y0 += 32768) {
                const unsigned ny = (unsigned)std::min(32768, G.nlaunch - y0);
                splitk_reduce_kernel<<<dim3(8, ny), 256, 0, st>>>(P->d_reds + G.first_launch + y0, P->d_xws, acc);
            }
            DMRG_CUDA(cudaGetLastError());
            if (P->timing) DMRG_CUDA(cudaEventRecord(P->ev[2 * gi + 1], st));
            continue;
        }
        for (int li = 0; li < G.nlaunch; li++) {   // more than one launch per group only with split_small (measurement aid)
            const PlanLaunch& L = P->launches[G.first_launch + li];
            int rc = launch_grouped_gemm(L.variant, P->copy_mode, P->d_segs, P->d_tiles + L.tile_begin, L.ntiles,
                                         P->ops->d_values, P->d_xws, P->d_psi_pad, acc, P->d_tmaps, st);
            if (rc != DMRG_OK) return rc;
        }
        if (P->timing) DMRG_CUDA(cudaEventRecord(P->ev[2 * gi + 1], st));
    }
    if (P->cplx) {
        for (int64_t y0 = 0; y0 < P->n_hd_blocks; y0 += 32768) {
            const unsigned ny = (unsigned)std::min<int64_t>(32768, P->n_hd_blocks - y0);
            sigma_z_finish_kernel<<<dim3(8, ny), 256, 0, st>>>(P->d_hd_blocks + y0, P->d_sigz, P->d_sigz + P->psi_size, sigma);
        }
        DMRG_CUDA(cudaGetLastError());
    }
    if (P->comm) { const int rc = comm_all_reduce(P->comm, sigma, P->psi_size, st); if (rc != DMRG_OK) return rc; }   // sharded plan: sum the partial sigmas
    if (P->timing) { DMRG_CUDA(cudaEventRecord(P->ev[2 * ng + 1], st)); P->timing_valid = true; }
    return DMRG_OK;
}

int dmrg_sigma_host(dmrg_plan* P, const double* psi_host, double* sigma_host, void* cuda_stream) {
    if (!P || !psi_host || !sigma_host) { set_error("dmrg_sigma_host: NULL argument"); return DMRG_EINVAL; }
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const size_t bytes = sizeof(double) * (size_t)P->psi_size;
    const size_t pad = (bytes + 255) & ~size_t(255);
    if (!P->d_host_io) DMRG_CUDA(cudaMalloc(&P->d_host_io, 2 * pad));   // staging vectors, kept for later calls
    double* d = P->d_host_io;
    double* d_sig = (double*)((char*)d + pad);
    DMRG_CUDA(cudaMemcpyAsync(d, psi_host, bytes, cudaMemcpyHostToDevice, st));
    int rc = dmrg_sigma(P, d, d_sig, cuda_stream);
    if (rc != DMRG_OK) return rc;
    DMRG_CUDA(cudaMemcpyAsync(sigma_host, d_sig, bytes, cudaMemcpyDeviceToHost, st));
    DMRG_CUDA(cudaStreamSynchronize(st));
    return DMRG_OK;
}

int dmrg_hdiag(dmrg_plan* P, double* diag, void* cuda_stream) {
    if (!P || !diag) { set_error("dmrg_hdiag: NULL argument"); return DMRG_EINVAL; }
    if (P->ops->structure_only) { set_error("dmrg_hdiag: the operator store was loaded without values (planning only)"); return DMRG_EINVAL; }
    cudaStream_t st = (cudaStream_t)cuda_stream;
    if (P->n_hd_tiles > 0 && P->cplx)
        hdiag_z_kernel<<<(unsigned)P->n_hd_tiles, 256, 0, st>>>(P->d_hd_blocks, P->d_hd_tiles, P->d_hd_items, P->ops->d_values, diag);
    else if (P->n_hd_tiles > 0)
        hdiag_kernel<<<(unsigned)P->n_hd_tiles, 256, 0, st>>>(P->d_hd_blocks, P->d_hd_tiles, P->d_hd_items, P->ops->d_values, diag);
    DMRG_CUDA(cudaGetLastError());
    if (P->comm) return comm_all_reduce(P->comm, diag, P->psi_size, st);
    return DMRG_OK;
}

}  // extern "C"
