/*
 * dmrg_sigma.h -- C ABI of the B200-native two-dot DMRG sigma-vector library.
 *
 * What it computes (arxiv/paper_2311_02854; line numbers are /root/reference/PAPER.md):
 *   sigma = H psi in the two-dot product space V_L x V_C1 x V_C2 x V_R, with H written as a
 *   sum of O(K^2) operator products  H = sum_mu O^L_mu O^C1_mu O^C2_mu O^R_mu   (Eq. 5),
 *     sigma[l'c1'c2'r'] = sum_mu sum_{l c1 c2 r} zeta [O^L]_{l'l} [O^C1]_{c1'c1} [O^C2]_{c2'c2}
 *                         [O^R]_{r'r} psi[l c1 c2 r]                               (Eq. 7)
 *   evaluated block by block over U(1)_N x U(1)_Sz symmetry sectors as
 *     X          = psi_blk * (O^R_blk)^T                                          (Eq. 11)
 *     sigma_blk += (c_mu zeta o1 o2) * O^L_blk * X                                (Eqs. 12-13)
 *   the dot factors being numbers for N,Sz symmetry, and called repeatedly by a
 *   Davidson eigensolver.
 *
 * Conventions:
 *   - All floating point data are IEEE FP64.  All matrices are dense ROW-MAJOR.
 *   - A sector is (N, 2Sz, dim).  An operator block O[row_sector, col_sector] is a
 *     dim[row] x dim[col] matrix; row sector = col sector + (dn, d2sz) of the operator.
 *   - Site (dot) basis: 0 vac, 1 beta, 2 alpha, 3 alpha-beta, (N,2Sz) = (0,0),(1,-1),(1,1),(2,0)
 *     (PAPER.md:49).
 *   - psi/sigma block (iL, c1, c2, iR) exists iff the four (N,2Sz) add up to the target; it is a
 *     dense row-major dim_L[iL] x dim_R[iR] matrix ("C order").  Blocks are stored
 *     back to back, sorted by (iR, c1, c2, iL), so all blocks sharing iR form one contiguous
 *     row panel.  dmrg_plan_psi_layout returns the table.
 *   - zeta = (-1)^{ p_C1 N_l + p_C2 (N_l+N_c1) + p_R (N_l+N_c1+N_c2) } with p_X the parity of the
 *     factor in slot X and N_x the particle numbers of the INPUT (ket) block (PAPER.md:73 names
 *     zeta without a formula; reading 3).
 *
 * Error behaviour: every int-returning entry point returns 0 on success and a negative
 * DMRG_E* code otherwise; dmrg_last_error() then returns a thread-local message.  No C++
 * exception crosses this boundary.  Nothing here falls back to a CPU path: without a CUDA
 * device every call that needs one fails with DMRG_ECUDA.
 *
 * Pointer kinds are stated per argument: [host] or [device].
 */
#ifndef DMRG_SIGMA_H
#define DMRG_SIGMA_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define DMRG_OK        0
#define DMRG_EINVAL   (-1)   /* bad argument / inconsistent tables            */
#define DMRG_ECHARGE  (-2)   /* a term does not conserve (N, 2Sz)              */
#define DMRG_ENOMEM   (-3)   /* host or device allocation failed               */
#define DMRG_ECUDA    (-4)   /* CUDA runtime error (text in dmrg_last_error)   */
#define DMRG_ENOCONV  (-5)   /* dmrg_davidson hit max_iter (outputs are valid) */

/* operator kinds, Eq. (19): {a+_p, A_pq, B_ps, P_pq, Q_ps, S_p, H}; LINCOMB is a
 * linear combination of one-index operators (the paper's "intermediates"). */
enum { DMRG_OP_H = 0, DMRG_OP_CRE = 1, DMRG_OP_A = 2, DMRG_OP_B = 3, DMRG_OP_P = 4, DMRG_OP_Q = 5,
       DMRG_OP_S = 6, DMRG_OP_LINCOMB = 7 };

typedef struct { int32_t n, two_sz, dim; } dmrg_sector;

typedef struct {
    int32_t side;         /* 0 = L, 1 = R                                                          */
    int32_t kind;         /* DMRG_OP_*; informational except DMRG_OP_LINCOMB                        */
    int32_t p, q;         /* spin-orbital labels (-1 unused); for LINCOMB p = row of lin_ptr        */
    int32_t dn, d2sz;     /* charge: row sector = col sector + (dn, d2sz); parity = dn & 1          */
    int64_t first_block;  /* index into blocks[]; ignored for LINCOMB                                */
    int32_t nblocks;      /* number of stored (non-zero) blocks; ignored for LINCOMB                 */
    int32_t reserved;
} dmrg_op_desc;

typedef struct { int32_t row_sector, col_sector; int64_t offset; } dmrg_block_desc; /* offset into values[] */

typedef struct {
    double  coef;            /* integral-derived coefficient c_mu                                   */
    int32_t op_l, trans_l;   /* operator id or -1 = identity; trans != 0 uses every block transposed */
    int32_t dot1, dot2;      /* ids into site_ops[]                                                  */
    int32_t op_r, trans_r;
} dmrg_term;

typedef struct { int32_t il, c1, c2, ir, dl, dr; int64_t offset; } dmrg_psi_block;

typedef struct dmrg_ops  dmrg_ops;    /* block-sparse operator store resident in HBM */
typedef struct dmrg_plan dmrg_plan;   /* GEMM-pair plan for one bond                  */

/* ---------------------------------------------------------------------------------------------
 * dmrg_ops_load: copy the block-sparse operator store {a+, A, B, P, Q, S, H}^{L,R} (Eq. 19-24,
 * PAPER.md:126-141, Fig. 1b "only the nonzero blocks are stored") into HBM and form the
 * linear-combination operators O = sum_s alpha_s a_s ("intermediates") on the device.
 *   secL/secR [host]  sector tables of the left / right renormalized basis
 *   ops       [host]  nops descriptors; the blocks of op i are blocks[first_block .. +nblocks)
 *   blocks    [host]  nblocks descriptors; at most one block per (op, row_sector)
 *   values    [host] or [device] (values_on_device != 0): nvalues doubles; block b is the row-major
 *             dim[row] x dim[col] matrix at values + blocks[b].offset.  Not retained: the store
 *             keeps its own (row-padded) copy, the caller may free `values` on return.
 *             values == NULL loads the STRUCTURE only (no CUDA call, no device memory): such a store
 *             can be planned (dmrg_plan_create, dmrg_plan_stat, dmrg_plan_psi_layout) to size a
 *             problem, but dmrg_sigma / dmrg_hdiag / dmrg_davidson on it fail with DMRG_EINVAL.
 *   lin_ptr   [host]  CSR over LINCOMB operators (nlin+1 entries); LINCOMB op with p = j is
 *             sum_{i in [lin_ptr[j], lin_ptr[j+1])} lin_coef[i] * ops[lin_op[i]]; all summands must be
 *             stored (non-LINCOMB) operators of the same side and charge as the LINCOMB op.
 * Ownership: *out owns its HBM; free with dmrg_ops_free.  Synchronous.
 */
int dmrg_ops_load(const dmrg_sector* secL, int32_t nsecL, const dmrg_sector* secR, int32_t nsecR,
                  const dmrg_op_desc* ops, int32_t nops,
                  const dmrg_block_desc* blocks, int64_t nblocks,
                  const double* values, int64_t nvalues, int32_t values_on_device,
                  const int64_t* lin_ptr, const int32_t* lin_op, const double* lin_coef, int32_t nlin,
                  dmrg_ops** out);
void    dmrg_ops_free(dmrg_ops* ops);
int64_t dmrg_ops_device_bytes(const dmrg_ops* ops);   /* HBM held by the store */

/* ---------------------------------------------------------------------------------------------
 * dmrg_plan_create: the "CPU preprocessing" of PAPER.md:97-99,145 -- expand every term mu and every
 * symmetry-block combination into GEMM pairs (Eq. 14), de-duplicate and merge the X = psi R^T
 * products, concatenate all contributions of one sigma block into one long-K GEMM in a fixed
 * order (the deterministic Eq. 13), tile, sort by cost, and upload the descriptors.
 *   terms      [host] nterms operator-pair terms (all four slots; identity = op -1 / site op 0..)
 *   site_ops   [host] nsite row-major 4x4 dot matrices; site_parity[i] = fermion parity of site op i
 *   n_total, two_sz_total: target quantum numbers of psi
 *   workspace_bytes: HBM the plan may use for the X intermediates (0 = default 8 GiB, raised to
 *              what the largest single term needs); terms are processed in chunks that fit it.
 *              The limit covers the X intermediates only: the split-K partial sigma tiles of a chunk live
 *              behind them in the same allocation (dmrg_plan_stat(16) = doubles actually allocated).
 *              Besides the workspace the plan owns a packed copy of the R-side blocks as stage 1 uses them
 *              (about the size of the R half of the store, twice where a block is used both ways) and a
 *              padded copy of psi; dmrg_plan_stat(8) reports the total.
 * Fails with DMRG_ECHARGE if a term does not conserve (N, 2Sz).  The plan borrows `ops`
 * (which must outlive it) and owns its descriptors and workspace.  Synchronous.
 *
 * dmrg_plan_create_opts: the same with every planner / kernel policy spelled out (there are no
 * environment variables).  Zero-initialise the struct for the defaults; fields:
 *   workspace_bytes    as above
 *   copy_mode          how operand tiles are staged global -> shared by the GEMM kernel:
 *                      0 = default (2); 1 = 16-byte cp.async (LDGSTS) issued by a 32-lane producer warp;
 *                      2 = TMA: one cp.async.bulk.tensor.2d per operand and pipeline stage through per-matrix
 *                      tensor maps the plan builds (the TMA unit zero-fills ragged tails)
 *   split_waves        split-K granularity of stage 2: a sigma block's K-loop is cut into parts no longer than
 *                      1/split_waves of the chunk's ideally balanced run time (0 = default 100)
 *   min_split_stages   ... but never shorter than this many GEMM_BK-wide pipeline stages (0 = default 96)
 *   max_merged_cols    widest N-merged stage-1 GEMM in columns (0 = default 4096)
 *   cost_order_only    1 = launch tiles in pure cost order; 0 (default) = inside a cost bucket, stage-2 tiles
 *                      follow (L sector of the sigma block, split-K part) so that they share L blocks in L2
 *   split_small        measurement aid for ncu (default 0 = off): tiles of jobs with min(M, N, K) < split_small
 *                      get a launch of their own (same tiles, same results, more launches)
 *   release_r_store    1 = after packing, free the store's R-side blocks (the plan's packed copy is then the only
 *                      one; the store can serve no further dmrg_plan_create); 0 = keep (default).  When the free
 *                      device memory does not hold the originals and the pack side by side, the R side is parked in
 *                      HOST memory (its size, pageable) and freed before the pack is allocated, and the pack is filled
 *                      from 4 GiB staging windows; 2 = always take that path.  (On that path the R side is given up
 *                      before the rest of the plan is allocated: if dmrg_plan_create then fails, e.g. DMRG_ENOMEM, the
 *                      store is left without its R side and must be loaded again.)
 *   tile_run_stages    stage 1: a CTA computes consecutive M tiles of one GEMM back to back (stage ring running on across
 *                      them) until it has this many pipeline stages of work, at most 8 tiles (0 = default 32; 1 = one
 *                      tile per CTA).  Same tiles and the same per-element summation order either way.
 *   shard_rank, shard_count   operator parallelism ("distribute operators and partition mu"): with
 *                      shard_count > 1 the plan evaluates only its share of the terms -- one contiguous range of the
 *                      planner's ordered term list (ordered by R operator, so a range needs only its own complementary
 *                      operators), cut where the running canonical cost crosses shard_rank/shard_count of the total;
 *                      every rank derives the same cuts from the same inputs.  dmrg_sigma / dmrg_hdiag then return
 *                      PARTIAL results: the caller sums them over ranks (one all-reduce of psi_size doubles per call;
 *                      paper_2311_02854_b200/sharded.py).  dmrg_plan_shard_terms lists the terms of the share.
 */
typedef struct {
    int64_t workspace_bytes;
    int32_t copy_mode;
    int32_t min_split_stages;
    double  split_waves;
    int32_t max_merged_cols;
    int32_t cost_order_only;
    int32_t split_small;
    int32_t release_r_store;
    int32_t shard_rank, shard_count;
    int32_t tile_run_stages;
    int32_t reserved[5];
} dmrg_plan_options;

int dmrg_plan_create(const dmrg_ops* ops, const dmrg_term* terms, int64_t nterms,
                     const double* site_ops, const int32_t* site_parity, int32_t nsite,
                     int32_t n_total, int32_t two_sz_total, int64_t workspace_bytes,
                     dmrg_plan** out);
int dmrg_plan_create_opts(const dmrg_ops* ops, const dmrg_term* terms, int64_t nterms,
                          const double* site_ops, const int32_t* site_parity, int32_t nsite,
                          int32_t n_total, int32_t two_sz_total, const dmrg_plan_options* options,
                          dmrg_plan** out);
void    dmrg_plan_destroy(dmrg_plan* plan);
int64_t dmrg_plan_psi_size(const dmrg_plan* plan);            /* doubles in psi / sigma         */
/* indices (into the caller's terms[]) of the terms this plan evaluates, in plan order; copies up to `capacity` of them
 * to out [host, may be NULL] and returns their number (= nterms unless the plan is a shard) */
int64_t dmrg_plan_shard_terms(const dmrg_plan* plan, int64_t* out, int64_t capacity);
int64_t dmrg_plan_num_psi_blocks(const dmrg_plan* plan);
int     dmrg_plan_psi_layout(const dmrg_plan* plan, dmrg_psi_block* out /* [host], num_psi_blocks */);

/* plan statistics, all per one dmrg_sigma call.  keys:
 *  0 tasks (term x block x dot transition)   1 algorithmic flops (2 dL dR dR' + 2 dL' dL dR' per task,
 *    identity factors cost 0 -- the paper's cost measure, Table 1 caption PAPER.md:151)
 *  2 executed stage-1 flops after de-duplication, unpadded    3 executed stage-2 flops, unpadded
 *  4 executed flops including tile padding                     5 stage-1 GEMM jobs   6 chunks
 *  7 kernel launches per sigma   8 device bytes held by the plan (descriptors + workspace)
 *  9 algorithmic operand bytes read per sigma (operator blocks once per use + X write/read + psi/sigma)
 * 10 stage-1 tiles   11 stage-2 tiles   12 canonical flops (= key 1 without de-duplication)
 * 13 executed flops with every segment's K padded to whole GEMM_BK(= 32)-wide pipeline stages
 * 14 the same with M and N padded to whole tiles as well; 15 ... padded to each tile's most loaded warp
 * 16 doubles allocated for the X workspace (X intermediates + split-K partial tiles of the largest chunk)
 * 17 tensor maps of the TMA path (one per operand matrix and orientation, 128 bytes each)
 * 18 / 19 mean fill of the stage-1 / stage-2 tiles (8 x 8 fragments used / 64)
 * 20 mean K per stage-1 tile   21 mean pipeline stages per stage-2 tile
 *                                           */
double  dmrg_plan_stat(const dmrg_plan* plan, int32_t key);

/* ---------------------------------------------------------------------------------------------
 * dmrg_sigma: sigma = H psi (Eq. 7).  psi, sigma [device], dmrg_plan_psi_size doubles each, must not
 * alias; sigma is OVERWRITTEN.  Work is enqueued on `cuda_stream` (a cudaStream_t, NULL = default
 * stream) and the call returns without synchronising.  Bitwise reproducible run to run: every
 * sigma element is accumulated by one thread block in plan order, no floating-point atomics.
 * A plan owns one X workspace and one padded copy of psi: calls on the same plan must be ordered (same stream,
 * or externally synchronised); use one plan per concurrent stream.
 * The call allocates nothing and never synchronises (per-stage timing off, no communicator attached): it may be issued
 * on a stream that is being captured into a CUDA graph, and the graph replayed (tests/test_gpu_parity.py).
 */
int dmrg_sigma(dmrg_plan* plan, const double* psi, double* sigma, void* cuda_stream);

/* dmrg_sigma_host: the same through HOST buffers (pageable or pinned): H2D copy of psi, dmrg_sigma,
 * D2H copy of sigma, synchronises.  Used for the end-to-end measurement. */
int dmrg_sigma_host(dmrg_plan* plan, const double* psi_host, double* sigma_host, void* cuda_stream);

/* dmrg_hdiag: diagonal of H in the psi layout ("diagonal part of Hamiltonian"), used as
 * the Davidson preconditioner.  diag [device], overwritten.  Asynchronous on `cuda_stream`. */
int dmrg_hdiag(dmrg_plan* plan, double* diag, void* cuda_stream);

/* ---------------------------------------------------------------------------------------------
 * dmrg_davidson: single-root Davidson (Ref. 74; parameters = DESIGN.md reading 11).
 *   x [device] in: initial guess (any non-zero norm), out: normalised Ritz vector.
 *   iteration k: w_k = H b_k (dmrg_sigma); G_ik = b_i.w_k; (theta, y) = lowest eigenpair of G;
 *   x = sum y_i b_i; r = sum y_i w_i - theta x; stop if |r| <= tol; t = r den/(den^2+delta^2),
 *   den = theta - Hd, delta = 1e-3; orthogonalise t against b_1..b_m (classical Gram-Schmidt twice),
 *   normalise -> b_{m+1}.  At m = max_space (>= 2) the basis collapses to {x} and H x is re-evaluated (that
 *   H psi counts as an iteration, as in the oracle).  One iteration = one H psi.  A zero initial guess is
 *   DMRG_EINVAL; a correction that vanishes after orthogonalisation ends the run (DMRG_ENOCONV, text says why).
 *   All vector work runs on the device; the host sees only O(m) scalars per iteration.
 *   thetas [host, may be NULL] receives theta_k for k < *iters (capacity max_iter).
 * Returns DMRG_OK if |r| <= tol, DMRG_ENOCONV if max_iter was reached (outputs still valid).
 * Synchronises `cuda_stream`.
 */
int dmrg_davidson(dmrg_plan* plan, double* x, int32_t max_iter, int32_t max_space, double tol,
                  double* energy, double* resid_norm, int32_t* iters, double* thetas,
                  void* cuda_stream);

/* ---------------------------------------------------------------------------------------------
 * Spin-orbit Hamiltonians: complex FP64, U(1)_N only, two-by-two dot blocks ("For relativistic Hamiltonian
 * including spin-orbit couplings, the spin projection is no longer a good quantum number, and [O]_{C1'C1} and [O]_{C2'C2}
 * can be either a scalar or a two-by-two matrix"; PAPER.md:285 names complex arithmetic as the extension).  The same
 * Eq. (7) in complex arithmetic:
 *   dmrg_ops_load_z    as dmrg_ops_load, with values [host or device] and lin_coef [host] holding (re, im) PAIRS of doubles
 *                      (numpy complex128): nvalues and dmrg_block_desc.offset count complex numbers.  Every sector label
 *                      and operator charge must have two_sz = d2sz = 0.  A "transposed" use of an operator (trans_l,
 *                      trans_r) means its conjugate transpose.  Store utilities (export, join, add_lincombs, derive) and
 *                      dmrg_renormalize refuse complex stores (DMRG_EINVAL).
 *   dmrg_plan_create_z as dmrg_plan_create_opts on such a store: coef_im [host, may be NULL = 0] the imaginary parts of the
 *                      term coefficients (real parts in terms[].coef); site_ops [host] nsite x 16 (re, im) pairs, row-major
 *                      4 x 4; only N is checked (DMRG_ECHARGE) and the two singly occupied site states (1 beta, 2 alpha)
 *                      belong to one dot sector, so a site matrix may connect them: such a two-by-two dot block is planned
 *                      as up to four (c', c) transitions per term and block, Eqs. (9)-(10) folded into the scalar factors.
 *   psi / sigma / diag of a complex plan are vectors of (re, im) pairs (complex128) in the psi layout;
 *   dmrg_plan_psi_size still counts DOUBLES (2 per number), dmrg_psi_block.offset counts numbers.  dmrg_sigma, dmrg_sigma_host,
 *   dmrg_hdiag (the real diagonal, written to both slots of every pair) and dmrg_davidson take such plans unchanged: a
 *   Hermitian H is a real symmetric operator on the 2n reals, with the same lowest eigenvalue, and every real eigenvector
 *   of it is a complex eigenvector of H.
 * How it runs (csrc/plan.cu): through the same real grouped FP64 GEMM kernel -- psi, X and sigma row-planar, the R blocks
 * packed as their real 2 x 2 images, the L blocks stored as theirs -- 8 M N K real flops per complex GEMM, the count of a
 * complex multiply-add, nothing computed twice.  The complex store takes 4 doubles per L-side entry (2 per R-side entry
 * plus 4 in the plan's packed copy). */
int dmrg_ops_load_z(const dmrg_sector* secL, int32_t nsecL, const dmrg_sector* secR, int32_t nsecR,
                    const dmrg_op_desc* ops, int32_t nops,
                    const dmrg_block_desc* blocks, int64_t nblocks,
                    const double* values, int64_t nvalues, int32_t values_on_device,
                    const int64_t* lin_ptr, const int32_t* lin_op, const double* lin_coef, int32_t nlin,
                    dmrg_ops** out);
int dmrg_plan_create_z(const dmrg_ops* ops, const dmrg_term* terms, const double* coef_im, int64_t nterms,
                       const double* site_ops, const int32_t* site_parity, int32_t nsite,
                       int32_t n_total, const dmrg_plan_options* options, dmrg_plan** out);
int32_t dmrg_ops_is_complex(const dmrg_ops* ops);
int32_t dmrg_plan_is_complex(const dmrg_plan* plan);

/* ---------------------------------------------------------------------------------------------
 * dmrg_dots_static: out[i] = sum_e V[i*stride + e] * w[e], i < m -- the block of dot products every Davidson
 * iteration needs (G_ik = b_i . w_k, the Gram-Schmidt coefficients, |r|^2; PAPER.md:162 keeps them on CPU rank 0),
 * for callers that cannot allocate device memory (CUDA graph capture, tight serving loops, harnesses that forbid
 * cudaMalloc).  Same two kernels, same fixed grid and summation tree as inside dmrg_davidson (bitwise the same
 * result for the same data), but the per-CTA partial sums live in a file-scope device array of
 * DMRG_DOTS_STATIC_MAX_VECTORS x 592 doubles (151552 bytes, held by every GPU that loads the library until exit)
 * instead of a cudaMalloc'ed workspace: the call makes no cudaMalloc / cudaFree and calls no allocating library routine.
 *   V [device] m vectors of n doubles, vector i at V + i*stride (stride >= n; ignored for m = 1); w [device] n doubles;
 *   out [device] m doubles, overwritten; m in [1, DMRG_DOTS_STATIC_MAX_VECTORS], else DMRG_EINVAL (the message names
 *   the limit); n >= 0 (n = 0 gives zeros).
 * Asynchronous on `cuda_stream`, on the current device.  All calls on one GPU share the one scratch array: calls that
 * may overlap on the GPU (different streams, no dependency between them) RACE on it -- keep them on one stream or
 * order them with events.  Every slot a call reads it has written itself, so nothing carries over between calls.
 */
#define DMRG_DOTS_STATIC_MAX_VECTORS 32
int dmrg_dots_static(const double* V, int64_t stride, int32_t m, const double* w, int64_t n, double* out,
                     void* cuda_stream);

/* ---------------------------------------------------------------------------------------------
 * dmrg_renormalize: the renormalization step that follows the Davidson step at every bond (Eq. 8),
 *     [O_new]_{r'r} = sum_{l'c'} sum_{lc} zeta A^{c'}_{l'r'} [O^blk]_{l'l} [O^site]_{c'c} A^{c}_{lr},
 * for every operator the enlarged block carries, evaluated block by block as Eqs. (15)-(18)
 * through the same grouped FP64 GEMM kernel as dmrg_sigma: Y = sum_terms (coef zeta o[c',c]) O^blk[L',L] A[(L c), R]
 * (Eqs. 15-16, one multi-segment GEMM per bra sub-block), then O_new[R',R] = A[., R']^T Y[., R] (Eqs. 17-18, the sum
 * over (L' C' L C) is the K-loop).  Deterministic, no atomics.
 *   in       the store of the block being enlarged (operators of side `side`, incl. the LINCOMB "intermediates"
 *            the terms use); borrowed, unchanged
 *   side     0: enlarged basis |l>|c> (a left block growing to the right), 1: |c>|r> (a right block growing left)
 *   new_sec  [host] sector table of the renormalized block
 *   wblocks  [host] the site tensor A (Eq. 3): block w is the row-major dim_old[old_sector] x
 *            dim_new[new_sector] matrix A[(l in old_sector, c = site_state), r in new_sector] at wvalues + offset;
 *            (N, 2Sz) of old_sector + site_state must equal those of new_sector; at most one block per triple
 *   wvalues  [host]
 *   new_ops  [host] descriptors of the operators to build (side is overwritten by `side`; kind, p, q are labels;
 *            dn, d2sz = the charge; first_block / nblocks ignored)
 *   term_ptr, terms [host] CSR: new operator k = sum_{t in [term_ptr[k], term_ptr[k+1])} coef_t * O^blk_t (x) o_t with
 *            O^blk_t = operator `op` of `in` (-1 = identity), every block transposed if trans != 0, and o_t =
 *            site_ops[site_op]; every term must carry the charge of its operator (else DMRG_ECHARGE).
 *            zeta is NOT part of coef: zeta = (-1)^{parity(second factor's operator) * N(ket of the first factor)},
 *            first/second = (block, site) for side 0, (site, block) for side 1 (reading 3, two factors)
 *   site_ops [host] nsite row-major 4x4 matrices, site_parity their fermion parities
 *   options  NULL = defaults: workspace_bytes (0 = 4 GiB) bounds the Y intermediates (new operators are processed in
 *            chunks), copy_mode as in dmrg_plan_options
 *   out      a new store holding the side-`side` operators new_ops[0..n) over new_sec (a block is present iff some
 *            term reaches it); owns its HBM, free with dmrg_ops_free
 *   stats    [host, may be NULL]
 * Enqueues on cuda_stream and synchronises it before returning.
 */
typedef struct { int32_t old_sector, site_state, new_sector, reserved; int64_t offset; } dmrg_wblock;
typedef struct { double coef; int32_t op, trans, site_op, reserved; } dmrg_rterm;
typedef struct { int64_t workspace_bytes; int32_t copy_mode; int32_t reserved[5]; } dmrg_renorm_options;
typedef struct { double flops, device_ms; int64_t launches, jobs, tiles, out_values, workspace_values, tensor_maps; } dmrg_renorm_stats;
int dmrg_renormalize(const dmrg_ops* in, int32_t side, const dmrg_sector* new_sec, int32_t n_new,
                     const dmrg_wblock* wblocks, int64_t n_wblocks, const double* wvalues, int64_t n_wvalues,
                     const dmrg_op_desc* new_ops, int32_t n_new_ops, const int64_t* term_ptr, const dmrg_rterm* terms,
                     const double* site_ops, const int32_t* site_parity, int32_t nsite,
                     const dmrg_renorm_options* options, void* cuda_stream, dmrg_ops** out, dmrg_renorm_stats* stats);

/* Store utilities a sweep needs around the renormalization step.
 * dmrg_ops_export: the store in the format dmrg_ops_load takes (unpadded row-major blocks): ops_out[num_ops] with
 *   first_block / nblocks filled, blocks_out[num_blocks], values_out[num_values], all [host]; LINCOMB operators are
 *   exported with the blocks they were formed into.  Synchronous.
 * dmrg_ops_sectors: copies up to `capacity` sectors of `side` to out (may be NULL); returns the sector count.
 * dmrg_ops_join: one two-sided store from a store with only side-0 operators and one with only side-1 operators
 *   (e.g. two dmrg_renormalize outputs).  No copy: *out takes over the device memory of both, which are consumed
 *   (freed as objects; do not use or free them afterwards).  Operator ids: left's, then right's shifted by
 *   dmrg_ops_num_ops(left).
 * dmrg_ops_add_lincombs: appends linear-combination operators O = sum_i coef_i op_i to a
 *   device-resident store; op_i = ops[lin_op[i]], or its transpose if lin_trans (may be NULL) has lin_trans[i] != 0
 *   (summands: existing operators of the same side whose charge, negated for a transposed summand, is the new
 *   operator's; CSR as in dmrg_ops_load, lin_ops[q].p = row of lin_ptr).  This is how the complementary operators
 *   are formed from the normal ones, P_pq = sum V (A_sr)^T, Q_pt = sum V B_qr + sum V (B_rq)^T (Eqs. 22-23,
 *   PAPER.md:135-137).  The new operators get ids num_ops, num_ops + 1, ...  Synchronous.
 * dmrg_ops_derive: the same linear combinations formed into a NEW store over the same sector tables (operator ids
 *   0 .. n_lin_ops-1, kinds as given); `src` is unchanged and can be freed afterwards -- e.g. keep {a+, S, H, P, Q}
 *   of a right block and drop its O(K^2) A and B operators. */
int64_t dmrg_ops_num_ops(const dmrg_ops* ops);
int64_t dmrg_ops_num_blocks(const dmrg_ops* ops);
int64_t dmrg_ops_num_values(const dmrg_ops* ops);
int     dmrg_ops_export(const dmrg_ops* ops, dmrg_op_desc* ops_out, dmrg_block_desc* blocks_out, double* values_out);
int     dmrg_ops_sectors(const dmrg_ops* ops, int32_t side, dmrg_sector* out, int32_t capacity);
int     dmrg_ops_join(dmrg_ops* left, dmrg_ops* right, dmrg_ops** out);
int     dmrg_ops_add_lincombs(dmrg_ops* ops, const dmrg_op_desc* lin_ops, int32_t n_lin_ops,
                              const int64_t* lin_ptr, const int32_t* lin_op, const double* lin_coef,
                              const int32_t* lin_trans, int32_t nlin);
int     dmrg_ops_derive(const dmrg_ops* src, const dmrg_op_desc* lin_ops, int32_t n_lin_ops,
                        const int64_t* lin_ptr, const int32_t* lin_op, const double* lin_coef,
                        const int32_t* lin_trans, int32_t nlin, dmrg_ops** out);

/* ---------------------------------------------------------------------------------------------
 * Operator parallelism over the GPUs of a node: the terms are partitioned over ranks
 * (dmrg_plan_options.shard_rank / shard_count) and the partial sigma vectors are summed with ONE all-reduce of psi_size
 * doubles per H psi (the paper: NCCL broadcast of the trial vector + reduce of sigma; here the Davidson vectors are
 * replicated and deterministic, so the broadcast is not needed).  One process per GPU:
 *   dmrg_comm_unique_id  rank 0: writes the NCCL unique id (returns its size in bytes, 128; id_out [host]); the caller
 *                        ships it to the other ranks (torch.distributed, MPI, a file)
 *   dmrg_comm_create     every rank, on its own device: ncclCommInitRank
 *   dmrg_plan_set_comm   attaches the communicator to a plan created as shard (rank, world): from then on dmrg_sigma and
 *                        dmrg_hdiag end with an in-place ncclAllReduce(SUM) on the caller's stream, right behind their
 *                        last launch, and return COMPLETE results on every rank; dmrg_davidson needs no change.
 *                        NULL detaches.  The plan borrows the communicator.
 * NCCL is loaded at run time (the libnccl.so.2 the process already has, e.g. torch's); without it these calls fail
 * with DMRG_ECUDA and everything single-GPU still works. */
typedef struct dmrg_comm dmrg_comm;
int  dmrg_comm_unique_id(void* id_out, int32_t capacity);
int  dmrg_comm_create(const void* id, int32_t rank, int32_t world, dmrg_comm** out);
void dmrg_comm_destroy(dmrg_comm* comm);
int  dmrg_plan_set_comm(dmrg_plan* plan, dmrg_comm* comm);

/* ---------------------------------------------------------------------------------------------
 * Per-stage device timing of the most recent dmrg_sigma with timing enabled (adds CUDA events
 * around each launch; off by default).  dmrg_plan_stage_ms synchronises and returns milliseconds:
 * which = 0 stage 1 (Eq. 11), 1 stage 2 + reduction (Eqs. 12-13), 2 whole call. */
int    dmrg_plan_set_timing(dmrg_plan* plan, int32_t enable);
double dmrg_plan_stage_ms(dmrg_plan* plan, int32_t which);

/* FP64 pipe micro-benchmarks used as the roofline denominator:
 * which = 0: dependent-free DFMA stream, 1: DMMA.8x8x4 (mma.sync m8n8k4 f64) stream.
 * Returns achieved TFLOP/s over `ms` milliseconds of back-to-back launches (>= 1 launch), or a
 * negative DMRG_E* code. */
double dmrg_fp64_peak_tflops(int32_t which, double ms, void* cuda_stream);

const char* dmrg_last_error(void);
const char* dmrg_version(void);

#ifdef __cplusplus
}
#endif
#endif /* DMRG_SIGMA_H */
