// dmrg_renormalize: the renormalization step of the sweep (Eq. 8; Eqs. 15-18) on the GPU,
// through the same grouped FP64 DMMA kernel as sigma = H psi, with the site tensor A in psi's place:
//   stage A (Eqs. 15-16):  Y_k[(L'C'), R] = sum_{terms t, (L C)} coef_t zeta o_t[C',C] . O_t[L',L] . A[(L C), R]
//                          one multi-segment GEMM per bra sub-block (L', C'): the K-loop walks the (term, ket
//                          sub-block) pairs in a fixed order; identity block factors are added in the tile prologue
//   stage B (Eqs. 17-18):  O_new_k[R', R] = A[., R']^T . Ycat_k[., R]        one GEMM per new block, K = the enlarged
//                          sector (all bra sub-blocks (L', C') stacked) -- the reduction of Eq. 18 is this K-loop
// Deterministic (no atomics), FP64.  Also here: the small store utilities a sweep needs around it
// (dmrg_ops_export, dmrg_ops_join, dmrg_ops_add_lincombs).
#include <algorithm>
#include <cmath>
#include <new>

#include "tmap.h"

namespace dmrg {

static const int R_SITE_N[4] = {0, 1, 1, 2};
static const int R_SITE_S[4] = {0, -1, 1, 0};

struct UnpackDesc { int64_t src, dst; int32_t rows, cols, ld, pad_; };
// dst[r*cols + c] = src[r*ld + c]      one CTA per block (the inverse of ops_store.cu's repack)
__global__ void __launch_bounds__(256) unpack_kernel(const UnpackDesc* __restrict__ desc, const double* __restrict__ src_base, double* __restrict__ dst_base) {
    const UnpackDesc d = desc[blockIdx.x];
    const int64_t n = (int64_t)d.rows * d.cols;
    for (int64_t e = threadIdx.x; e < n; e += blockDim.x) {
        const int r = (int)(e / d.cols), c = (int)(e - (int64_t)r * d.cols);
        dst_base[d.dst + e] = src_base[d.src + (int64_t)r * d.ld + c];
    }
}

struct LinDesc2 { int64_t dst; int32_t rows, cols, ld, pad_; int32_t sum_begin, sum_end; };   // dst block: rows x cols, row pitch ld
struct LinSummand2 { int64_t src; double coef; int32_t present, trans, ld_src, pad_; };   // trans: the summand's block is used transposed
// dst[i][j] = sum_s coef_s * (trans_s ? src_s[j][i] : src_s[i][j])  in summand order (deterministic); row pads are written as zeros.
// The same arithmetic as ops_store.cu's lincomb_kernel, plus transposed summands (P_pq = sum V (A_sr)^T, Q_pt = sum V B_qr + sum V (B_rq)^T:
// the complementary operators from the normal ones, SURVEY.md section 8.0 identity I5).      grid (chunks, blocks)
__global__ void __launch_bounds__(256) lincomb2_kernel(const LinDesc2* __restrict__ desc, const LinSummand2* __restrict__ sums, double* __restrict__ vals) {
    const LinDesc2 d = desc[blockIdx.y];
    const int64_t n = (int64_t)d.rows * d.ld;
    for (int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; e < n; e += (int64_t)gridDim.x * blockDim.x) {
        const int i = (int)(e / d.ld), j = (int)(e - (int64_t)i * d.ld);
        double acc = 0.0;
        if (j < d.cols)
            for (int q = d.sum_begin; q < d.sum_end; q++) {
                const LinSummand2 s = sums[q];
                if (s.present) acc = fma(s.coef, s.trans ? vals[s.src + (int64_t)j * s.ld_src + i] : vals[s.src + (int64_t)i * s.ld_src + j], acc);
            }
        vals[d.dst + e] = acc;
    }
}
constexpr int64_t kAbsent = -1;   // row_off of an absent block (offsets of present blocks are >= 0: stores are rebased to their lowest allocation)

// make `new_base` (<= every allocation of the store) the origin of the store's offsets
static void rebase(dmrg_ops* S, double* new_base) {
    const int64_t shift = (int64_t)(S->d_values - new_base);
    if (shift == 0) return;
    for (auto& ro : S->row_off)
        for (auto& o : ro)
            if (o >= 0) o += shift;
    S->d_values = new_base;
}

static int find_sec(const std::vector<dmrg_sector>& s, int n, int two_sz) {
    for (size_t i = 0; i < s.size(); i++)
        if (s[i].n == n && s[i].two_sz == two_sz) return (int)i;
    return -1;
}

template <typename T>
static int upload(T** dptr, const std::vector<T>& v) {
    DMRG_CUDA(cudaMalloc((void**)dptr, std::max<size_t>(v.size() * sizeof(T), 16)));
    if (!v.empty()) DMRG_CUDA(cudaMemcpy(*dptr, v.data(), v.size() * sizeof(T), cudaMemcpyHostToDevice));
    return DMRG_OK;
}

struct RenormScratch {   // transient device buffers of one dmrg_renormalize call
    Seg* d_segs = nullptr; TileDesc* d_tiles = nullptr; TensorMap* d_tmaps = nullptr;
    double *d_w = nullptr, *d_y = nullptr;
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    ~RenormScratch() {
        cudaFree(d_segs); cudaFree(d_tiles); cudaFree(d_tmaps); cudaFree(d_w); cudaFree(d_y);
        if (e0) cudaEventDestroy(e0);
        if (e1) cudaEventDestroy(e1);
    }
};

static int renormalize_impl(const dmrg_ops* in, int side, const dmrg_sector* new_sec, int n_new, const dmrg_wblock* wb, int64_t n_wb,
                            const double* wvalues, int64_t n_wvalues, const dmrg_op_desc* new_ops, int n_new_ops, const int64_t* term_ptr,
                            const dmrg_rterm* terms, const double* site_ops, const int32_t* site_parity, int nsite,
                            const dmrg_renorm_options* opt, cudaStream_t st, dmrg_ops* out, dmrg_renorm_stats* stats) {
    DMRG_REQUIRE(in && !in->structure_only, "dmrg_renormalize: the input store has no values");
    DMRG_REQUIRE(!in->r_released, "dmrg_renormalize: the R-side blocks of the input store were released to a plan");
    DMRG_REQUIRE(side == 0 || side == 1, "dmrg_renormalize: side must be 0 (block x site) or 1 (site x block)");
    DMRG_REQUIRE(new_sec && n_new > 0 && wb && n_wb > 0 && wvalues && new_ops && n_new_ops > 0 && term_ptr && site_ops && site_parity && nsite > 0,
                 "dmrg_renormalize: NULL or empty argument");
    const auto& secO = in->sec[side];
    const int nO = (int)secO.size();
    DMRG_REQUIRE(nO > 0, "dmrg_renormalize: the input store has no sectors on side %d", side);
    const int nops_in = (int)in->ops.size();
    const int copy_mode = (opt && (opt->copy_mode == COPY_LDGSTS || opt->copy_mode == COPY_TMA)) ? opt->copy_mode : COPY_TMA;
    const int64_t ws_elems = ((opt && opt->workspace_bytes > 0) ? opt->workspace_bytes : (int64_t(4) << 30)) / 8;
    const int TILE = kVariants[0].bm;

    // ---- the site tensor A: sub-blocks (old sector, site state) -> new sector, stacked per new sector -----
    struct Sub { int i_old, n_site; int64_t row0; int64_t src; };
    std::vector<std::vector<Sub>> sub(n_new);
    std::vector<int64_t> enl(n_new, 0), woff(n_new, 0);
    std::vector<int> ldw(n_new);
    for (int r = 0; r < n_new; r++) { DMRG_REQUIRE(new_sec[r].dim > 0, "dmrg_renormalize: new sector %d has dim <= 0", r); ldw[r] = (int)round_up2(new_sec[r].dim); }
    for (int64_t w = 0; w < n_wb; w++) {
        const dmrg_wblock& b = wb[w];
        DMRG_REQUIRE(b.old_sector >= 0 && b.old_sector < nO && b.site_state >= 0 && b.site_state < 4 && b.new_sector >= 0 && b.new_sector < n_new,
                     "dmrg_renormalize: site-tensor block %lld: index out of range", (long long)w);
        const dmrg_sector& so = secO[b.old_sector];
        DMRG_REQUIRE(so.n + R_SITE_N[b.site_state] == new_sec[b.new_sector].n && so.two_sz + R_SITE_S[b.site_state] == new_sec[b.new_sector].two_sz,
                     "dmrg_renormalize: site-tensor block %lld does not conserve (N, 2Sz)", (long long)w);
        DMRG_REQUIRE(b.offset >= 0 && b.offset + (int64_t)so.dim * new_sec[b.new_sector].dim <= n_wvalues, "dmrg_renormalize: site-tensor block %lld exceeds wvalues[]", (long long)w);
        for (const Sub& s : sub[b.new_sector])
            DMRG_REQUIRE(!(s.i_old == b.old_sector && s.n_site == b.site_state), "dmrg_renormalize: site-tensor block %lld given twice", (long long)w);
        sub[b.new_sector].push_back({b.old_sector, b.site_state, enl[b.new_sector], b.offset});
        enl[b.new_sector] += so.dim;
    }
    int64_t wtop = 0;
    for (int r = 0; r < n_new; r++) { woff[r] = wtop; wtop += enl[r] * ldw[r]; }
    std::vector<double> hw((size_t)std::max<int64_t>(wtop, 2), 0.0);
    for (int r = 0; r < n_new; r++)
        for (const Sub& s : sub[r]) {
            const int d = secO[s.i_old].dim, k = new_sec[r].dim;
            for (int a = 0; a < d; a++)
                std::copy(wvalues + s.src + (int64_t)a * k, wvalues + s.src + (int64_t)(a + 1) * k, hw.begin() + woff[r] + (s.row0 + a) * ldw[r]);
        }

    // ---- validate the terms; per-op inverse sector map of the input store -----------------------------------
    std::vector<std::vector<int32_t>> rowof(nops_in);
    for (int o = 0; o < nops_in; o++) {
        if (in->ops[o].side != side) continue;
        const int ns = (int)in->colsec[o].size();
        rowof[o].assign(ns, -1);
        for (int r = 0; r < ns; r++)
            if (in->colsec[o][r] >= 0) rowof[o][in->colsec[o][r]] = r;
    }
    for (int k = 0; k < n_new_ops; k++) {
        DMRG_REQUIRE(term_ptr[k] <= term_ptr[k + 1], "dmrg_renormalize: term_ptr not monotone");
        for (int64_t t = term_ptr[k]; t < term_ptr[k + 1]; t++) {
            const dmrg_rterm& T = terms[t];
            DMRG_REQUIRE(T.op >= -1 && T.op < nops_in && (T.op < 0 || in->ops[T.op].side == side), "dmrg_renormalize: term %lld: bad block operator id", (long long)t);
            DMRG_REQUIRE(T.site_op >= 0 && T.site_op < nsite, "dmrg_renormalize: term %lld: bad site operator id", (long long)t);
            int dn = 0, ds = 0;
            if (T.op >= 0) { const int sg = T.trans ? -1 : 1; dn = sg * in->ops[T.op].dn; ds = sg * in->ops[T.op].d2sz; }
            const double* o = site_ops + 16 * (size_t)T.site_op;
            for (int a = 0; a < 4; a++)
                for (int b = 0; b < 4; b++)
                    if (o[4 * a + b] != 0.0 && (dn + R_SITE_N[a] - R_SITE_N[b] != new_ops[k].dn || ds + R_SITE_S[a] - R_SITE_S[b] != new_ops[k].d2sz)) {
                        set_error("dmrg_renormalize: term %lld of new operator %d does not carry the operator's charge (%d, %d)", (long long)t, k, new_ops[k].dn, new_ops[k].d2sz);
                        return DMRG_ECHARGE;
                    }
        }
    }
    auto blk_off = [&](int op, int trans, int i_bra, int i_ket) -> int64_t {   // offset of O[i_bra, i_ket] as used, or kAbsent
        if (!trans) return in->colsec[op][i_bra] == i_ket ? in->row_off[op][i_bra] : kAbsent;
        return in->colsec[op][i_ket] == i_bra ? in->row_off[op][i_ket] : kAbsent;
    };

    // ---- output store layout + job lists, new operators processed in chunks that fit the Y workspace ------
    out->sec[side].assign(new_sec, new_sec + n_new);
    out->ops.assign(new_ops, new_ops + n_new_ops);
    out->row_off.assign(n_new_ops, std::vector<int64_t>(n_new, -1));
    out->colsec.assign(n_new_ops, std::vector<int32_t>(n_new, -1));
    std::vector<Job> jobs;
    std::vector<Seg> segs;
    std::vector<Tile> tiles;
    struct Launch { int64_t tile_begin, ntiles; };
    std::vector<Launch> launches;   // alternating stage A, stage B per chunk
    MapTable maps;
    int64_t top = 0, ytop = 0, ypeak = 0;
    double flops = 0.0;
    struct TileRec { Tile t; double cost; };
    std::vector<TileRec> recA, recB;
    std::vector<std::pair<int, int>> cut_m, cut_n;
    auto flush = [&]() {
        for (auto* rec : {&recA, &recB}) {
            std::stable_sort(rec->begin(), rec->end(), [](const TileRec& a, const TileRec& b) { return a.cost > b.cost; });
            launches.push_back({(int64_t)tiles.size(), (int64_t)rec->size()});
            for (auto& r : *rec) tiles.push_back(r.t);
            rec->clear();
        }
        ypeak = std::max(ypeak, ytop);
        ytop = 0;
    };
    for (int k = 0; k < n_new_ops; k++) {
        dmrg_op_desc& od = out->ops[k];
        od.side = side;
        od.first_block = 0; od.nblocks = 0;
        for (int r = 0; r < n_new; r++) out->colsec[k][r] = find_sec(out->sec[side], new_sec[r].n - od.dn, new_sec[r].two_sz - od.d2sz);
        for (int r = 0; r < n_new; r++) {   // ket sector r, bra sector rb = r + charge
            const int rb = find_sec(out->sec[side], new_sec[r].n + od.dn, new_sec[r].two_sz + od.d2sz);
            if (rb < 0) continue;
            const int dk = new_sec[r].dim, dkb = new_sec[rb].dim;
            const int ldy = (int)round_up2(dk);
            const int64_t ysize = enl[rb] * ldy;
            // segments of every bra sub-block first: the block exists iff some term reaches it
            struct PendJob { const Sub* sb; std::vector<Seg> ident, gemm; };
            std::vector<PendJob> pend;
            bool any = false;
            for (const Sub& sb : sub[rb]) {
                PendJob pj{&sb, {}, {}};
                for (int64_t t = term_ptr[k]; t < term_ptr[k + 1]; t++) {
                    const dmrg_rterm& T = terms[t];
                    const double* o = site_ops + 16 * (size_t)T.site_op;
                    const int p_site = site_parity[T.site_op] & 1;
                    const int p_blk = T.op >= 0 ? (in->ops[T.op].dn & 1) : 0;
                    for (const Sub& sk : sub[r]) {
                        const double oc = o[4 * sb.n_site + sk.n_site];
                        if (oc == 0.0) continue;
                        int64_t a_off = kAbsent;
                        if (T.op < 0) { if (sb.i_old != sk.i_old) continue; }
                        else { a_off = blk_off(T.op, T.trans != 0, sb.i_old, sk.i_old); if (a_off < 0) continue; }
                        const int zexp = side == 0 ? p_site * secO[sk.i_old].n : p_blk * R_SITE_N[sk.n_site];
                        Seg s;
                        s.alpha = T.coef * ((zexp & 1) ? -1.0 : 1.0) * oc;
                        s.K = secO[sk.i_old].dim;
                        s.flags = (SP_PSI << SEG_B_SPACE_SHIFT);
                        s.b_off = woff[r] + sk.row0 * ldw[r]; s.ldb = ldw[r];
                        s.a_map = s.b_map = 0; s.a_o0 = 0; s.a_pitch = s.b_pitch = 0; s.a_bytes = s.b_bytes = 0;
                        if (T.op < 0) { s.a_off = 0; s.lda = 0; s.flags |= SEG_A_IDENT; pj.ident.push_back(s); }
                        else {
                            const int dbra = secO[sb.i_old].dim, dket = secO[sk.i_old].dim;
                            s.a_off = a_off; s.lda = (int)round_up2(T.trans ? dbra : dket);
                            s.flags |= (SP_OPS << SEG_A_SPACE_SHIFT) | (T.trans ? SEG_A_MCONTIG : 0);
                            const BoxShape ba = box_shape(T.trans ? 1 : 0, dket, dbra, TILE);
                            s.a_map = T.trans ? maps.get(MS_OPS, a_off, 1, dbra, dket, s.lda, ba) : maps.get(MS_OPS, a_off, 0, dket, dbra, s.lda, ba);
                            s.a_pitch = (uint16_t)ba.inner; s.a_bytes = 8u * ba.inner * ba.outer;
                            const BoxShape bb = box_shape(1, dket, dk, TILE);
                            s.b_map = maps.get(MS_PSI, s.b_off, 1, dk, dket, ldw[r], bb);
                            s.b_pitch = (uint16_t)bb.inner; s.b_bytes = 8u * bb.inner * bb.outer;
                            pj.gemm.push_back(s);
                            flops += 2.0 * dbra * dket * dk;
                        }
                        any = true;
                    }
                }
                pend.push_back(std::move(pj));
            }
            if (!any) continue;
            if (ytop + ysize > ws_elems && ytop > 0) flush();
            const int64_t y_off = ytop;
            ytop += ysize;
            out->row_off[k][rb] = top;
            od.nblocks++;
            // stage A jobs: one per bra sub-block (a sub-block no term reaches is written as zeros: a job without segments)
            for (PendJob& pj : pend) {
                Job jb;
                jb.c_off = y_off + pj.sb->row0 * ldy; jb.ldc = ldy; jb.M = secO[pj.sb->i_old].dim; jb.N = dk;
                jb.flags = (SP_X << JOB_C_SPACE_SHIFT);
                jb.seg_begin = (int32_t)segs.size();
                segs.insert(segs.end(), pj.ident.begin(), pj.ident.end());
                segs.insert(segs.end(), pj.gemm.begin(), pj.gemm.end());
                jb.seg_end = (int32_t)segs.size();
                jb.nstages = 0;
                for (const Seg& s : pj.gemm) jb.nstages += (s.K + GEMM_BK - 1) / GEMM_BK;
                cut_dim(jb.M, TILE, cut_m);
                cut_dim(jb.N, TILE, cut_n);
                for (auto& a : cut_m)
                    for (auto& b : cut_n) recA.push_back({{(int32_t)jobs.size(), a.first, b.first, (uint16_t)a.second, (uint16_t)b.second}, jb.nstages + 1.0});
                jobs.push_back(jb);
            }
            // stage B job: O_new[rb, r] = W[rb]^T Ycat
            {
                Seg s;
                s.alpha = 1.0; s.K = (int32_t)enl[rb];
                s.a_off = woff[rb]; s.lda = ldw[rb];
                s.b_off = y_off; s.ldb = ldy;
                s.flags = (SP_PSI << SEG_A_SPACE_SHIFT) | SEG_A_MCONTIG | (SP_X << SEG_B_SPACE_SHIFT);
                const BoxShape ba = box_shape(1, (int)enl[rb], dkb, TILE), bb = box_shape(1, (int)enl[rb], dk, TILE);
                s.a_map = maps.get(MS_PSI, woff[rb], 1, dkb, enl[rb], ldw[rb], ba);
                s.b_map = maps.get(MS_X, y_off, 1, dk, enl[rb], ldy, bb);
                s.a_o0 = 0; s.a_pitch = (uint16_t)ba.inner; s.b_pitch = (uint16_t)bb.inner;
                s.a_bytes = 8u * ba.inner * ba.outer; s.b_bytes = 8u * bb.inner * bb.outer;
                Job jb;
                jb.c_off = top; jb.ldc = ldy; jb.M = dkb; jb.N = dk;
                jb.flags = (SP_SIGMA << JOB_C_SPACE_SHIFT);
                jb.seg_begin = (int32_t)segs.size(); jb.seg_end = jb.seg_begin + 1;
                jb.nstages = (int32_t)((enl[rb] + GEMM_BK - 1) / GEMM_BK);
                segs.push_back(s);
                cut_dim(jb.M, TILE, cut_m);
                cut_dim(jb.N, TILE, cut_n);
                for (auto& a : cut_m)
                    for (auto& b : cut_n) recB.push_back({{(int32_t)jobs.size(), a.first, b.first, (uint16_t)a.second, (uint16_t)b.second}, jb.nstages + 1.0});
                jobs.push_back(jb);
                flops += 2.0 * dkb * (double)enl[rb] * dk;
            }
            top += (int64_t)dkb * ldy;
            DMRG_REQUIRE(segs.size() < ((size_t)1 << 31) && jobs.size() < ((size_t)1 << 31), "dmrg_renormalize: descriptor table overflow");
        }
    }
    flush();
    for (Seg& sg : segs) sg.flags |= sg.alpha == 1.0 ? SEG_ALPHA_ONE : (sg.alpha == -1.0 ? SEG_ALPHA_NEG : 0u);

    // ---- device: allocate, upload, run ---------------------------------------------------------------------------
    out->nvalues_dev = top;
    out->device_bytes = sizeof(double) * (size_t)std::max<int64_t>(top, 2);
    DMRG_CUDA(cudaMalloc(&out->d_values, (size_t)out->device_bytes));
    out->owned.push_back(out->d_values);
    DMRG_CUDA(cudaMemsetAsync(out->d_values, 0, (size_t)out->device_bytes, st));   // row pads must be zero
    RenormScratch sc;
    int rc;
    DMRG_CUDA(cudaMalloc(&sc.d_w, sizeof(double) * hw.size()));
    DMRG_CUDA(cudaMemcpyAsync(sc.d_w, hw.data(), sizeof(double) * hw.size(), cudaMemcpyHostToDevice, st));
    DMRG_CUDA(cudaMalloc(&sc.d_y, sizeof(double) * (size_t)std::max<int64_t>(ypeak, 2)));
    if ((rc = upload(&sc.d_segs, segs))) return rc;
    if ((rc = upload(&sc.d_tiles, make_tile_descs(tiles, jobs, segs)))) return rc;
    {
        double* const base[4] = {in->d_values, sc.d_y, sc.d_w, nullptr};
        std::vector<TensorMap> tm;
        if ((rc = encode_tensor_maps(maps.descs, base, tm))) return rc;
        if ((rc = upload(&sc.d_tmaps, tm))) return rc;
    }
    if ((rc = gemm_init())) return rc;
    DMRG_CUDA(cudaEventCreate(&sc.e0));
    DMRG_CUDA(cudaEventCreate(&sc.e1));
    DMRG_CUDA(cudaEventRecord(sc.e0, st));
    int nlaunch = 0;
    for (const Launch& L : launches) {
        if (L.ntiles == 0) continue;
        if ((rc = launch_grouped_gemm(0, copy_mode, sc.d_segs, sc.d_tiles + L.tile_begin, L.ntiles, in->d_values, sc.d_y, sc.d_w, out->d_values, sc.d_tmaps, st)))
            return rc;
        nlaunch++;
    }
    DMRG_CUDA(cudaEventRecord(sc.e1, st));
    DMRG_CUDA(cudaStreamSynchronize(st));   // the scratch buffers die with this call
    if (stats) {
        float ms = 0.f;
        cudaEventElapsedTime(&ms, sc.e0, sc.e1);
        stats->flops = flops; stats->device_ms = ms; stats->launches = nlaunch; stats->jobs = (int64_t)jobs.size();
        stats->tiles = (int64_t)tiles.size(); stats->out_values = top; stats->workspace_values = ypeak; stats->tensor_maps = (int64_t)maps.descs.size();
    }
    return DMRG_OK;
}

}  // namespace dmrg

using namespace dmrg;

extern "C" {

int dmrg_renormalize(const dmrg_ops* in, int32_t side, const dmrg_sector* new_sec, int32_t n_new, const dmrg_wblock* wblocks, int64_t n_wblocks,
                     const double* wvalues, int64_t n_wvalues, const dmrg_op_desc* new_ops, int32_t n_new_ops, const int64_t* term_ptr,
                     const dmrg_rterm* terms, const double* site_ops, const int32_t* site_parity, int32_t nsite,
                     const dmrg_renorm_options* options, void* cuda_stream, dmrg_ops** out, dmrg_renorm_stats* stats) {
    if (!out) { set_error("dmrg_renormalize: out is NULL"); return DMRG_EINVAL; }
    *out = nullptr;
    if (in && in->cplx) { set_error("%s: complex stores (dmrg_ops_load_z) are served by dmrg_plan_create_z / dmrg_sigma / dmrg_hdiag / dmrg_davidson only", "dmrg_renormalize"); return DMRG_EINVAL; }
    dmrg_ops* S = new (std::nothrow) dmrg_ops();
    if (!S) { set_error("dmrg_renormalize: out of host memory"); return DMRG_ENOMEM; }
    int rc;
    try {
        rc = renormalize_impl(in, side, new_sec, n_new, wblocks, n_wblocks, wvalues, n_wvalues, new_ops, n_new_ops, term_ptr, terms, site_ops, site_parity,
                              nsite, options, (cudaStream_t)cuda_stream, S, stats);
    } catch (const std::bad_alloc&) {
        set_error("dmrg_renormalize: out of host memory");
        rc = DMRG_ENOMEM;
    } catch (const std::exception& e) {
        set_error("dmrg_renormalize: %s", e.what());
        rc = DMRG_EINVAL;
    }
    if (rc != DMRG_OK) { dmrg_ops_free(S); return rc; }
    *out = S;
    return DMRG_OK;
}

int64_t dmrg_ops_num_ops(const dmrg_ops* S) { return S ? (int64_t)S->ops.size() : 0; }

int64_t dmrg_ops_num_blocks(const dmrg_ops* S) {
    if (!S) return 0;
    int64_t n = 0;
    for (size_t o = 0; o < S->ops.size(); o++)
        for (size_t r = 0; r < S->row_off[o].size(); r++) n += (S->row_off[o][r] >= 0) ? 1 : 0;
    return n;
}

int64_t dmrg_ops_num_values(const dmrg_ops* S) {
    if (!S) return 0;
    int64_t n = 0;
    for (size_t o = 0; o < S->ops.size(); o++) {
        const auto& sec = S->sec[S->ops[o].side];
        for (size_t r = 0; r < S->row_off[o].size(); r++)
            if ((S->row_off[o][r] >= 0)) n += (int64_t)sec[r].dim * sec[S->colsec[o][r]].dim;
    }
    return n;
}

int dmrg_ops_export(const dmrg_ops* S, dmrg_op_desc* ops_out, dmrg_block_desc* blocks_out, double* values_out) {
    if (!S || !ops_out || !blocks_out || !values_out) { set_error("dmrg_ops_export: NULL argument"); return DMRG_EINVAL; }
    if (S->structure_only) { set_error("dmrg_ops_export: the store was loaded without values"); return DMRG_EINVAL; }
    if (S->cplx) { set_error("%s: complex stores (dmrg_ops_load_z) are served by dmrg_plan_create_z / dmrg_sigma / dmrg_hdiag / dmrg_davidson only", "dmrg_ops_export"); return DMRG_EINVAL; }
    if (S->r_released) { set_error("dmrg_ops_export: the R-side blocks of this store were released to a plan"); return DMRG_EINVAL; }
    std::vector<UnpackDesc> desc;
    int64_t nb = 0, nv = 0;
    for (size_t o = 0; o < S->ops.size(); o++) {
        const auto& sec = S->sec[S->ops[o].side];
        ops_out[o] = S->ops[o];
        ops_out[o].first_block = nb;
        int cnt = 0;
        for (size_t r = 0; r < S->row_off[o].size(); r++) {
            if (!(S->row_off[o][r] >= 0)) continue;
            const int c = S->colsec[o][r];
            blocks_out[nb] = {(int32_t)r, c, nv};
            desc.push_back({S->row_off[o][r], nv, sec[r].dim, sec[c].dim, (int32_t)round_up2(sec[c].dim), 0});
            nv += (int64_t)sec[r].dim * sec[c].dim;
            nb++; cnt++;
        }
        ops_out[o].nblocks = cnt;
    }
    if (nv == 0) return DMRG_OK;
    double* d_flat = nullptr;
    UnpackDesc* d_desc = nullptr;
    DMRG_CUDA(cudaMalloc(&d_flat, sizeof(double) * (size_t)nv));
    cudaError_t e = cudaMalloc(&d_desc, sizeof(UnpackDesc) * desc.size());
    if (e == cudaSuccess) e = cudaMemcpy(d_desc, desc.data(), sizeof(UnpackDesc) * desc.size(), cudaMemcpyHostToDevice);
    if (e == cudaSuccess) {
        for (size_t i = 0; i < desc.size(); i += 65535 * 16) {
            const unsigned n = (unsigned)std::min<size_t>(desc.size() - i, 65535 * 16);
            unpack_kernel<<<n, 256>>>(d_desc + i, S->d_values, d_flat);
        }
        e = cudaGetLastError();
    }
    if (e == cudaSuccess) e = cudaMemcpy(values_out, d_flat, sizeof(double) * (size_t)nv, cudaMemcpyDeviceToHost);
    cudaFree(d_flat);
    cudaFree(d_desc);
    if (e != cudaSuccess) { set_error("dmrg_ops_export: %s", cudaGetErrorString(e)); return DMRG_ECUDA; }
    return DMRG_OK;
}

int dmrg_ops_sectors(const dmrg_ops* S, int32_t side, dmrg_sector* out, int32_t capacity) {
    if (!S || (side != 0 && side != 1)) { set_error("dmrg_ops_sectors: bad argument"); return DMRG_EINVAL; }
    const int n = (int)S->sec[side].size();
    if (out) std::copy(S->sec[side].begin(), S->sec[side].begin() + std::min(n, (int)capacity), out);
    return n;
}

int dmrg_ops_join(dmrg_ops* left, dmrg_ops* right, dmrg_ops** out) {
    if (!left || !right || !out) { set_error("dmrg_ops_join: NULL argument"); return DMRG_EINVAL; }
    *out = nullptr;
    if (left->cplx || right->cplx) { set_error("%s: complex stores (dmrg_ops_load_z) are served by dmrg_plan_create_z / dmrg_sigma / dmrg_hdiag / dmrg_davidson only", "dmrg_ops_join"); return DMRG_EINVAL; }
    if (left->structure_only || right->structure_only || left->owned.empty() || right->owned.empty()) { set_error("dmrg_ops_join: both stores must hold device values"); return DMRG_EINVAL; }
    if (!left->sec[1].empty() || !right->sec[0].empty() || left->sec[0].empty() || right->sec[1].empty()) {
        set_error("dmrg_ops_join: `left` must hold only side-0 operators and `right` only side-1 operators");
        return DMRG_EINVAL;
    }
    dmrg_ops* J = new (std::nothrow) dmrg_ops();
    if (!J) { set_error("dmrg_ops_join: out of host memory"); return DMRG_ENOMEM; }
    const size_t nr = right->ops.size();
    // one address space: offsets relative to the lower of the two bases (both cudaMalloc'ed: the difference is a
    // multiple of 32 doubles, so 16-byte alignment of every row is preserved)
    double* base = std::min(left->d_values, right->d_values);
    rebase(left, base);
    rebase(right, base);
    J->sec[0] = left->sec[0];
    J->sec[1] = right->sec[1];
    J->ops = left->ops;
    J->ops.insert(J->ops.end(), right->ops.begin(), right->ops.end());
    J->row_off = left->row_off;
    J->colsec = left->colsec;
    for (size_t o = 0; o < nr; o++) {
        J->colsec.push_back(right->colsec[o]);
        J->row_off.push_back(right->row_off[o]);
    }
    J->d_values = base;
    // release_r_store needs the R side in ONE allocation of its own: true when `right` is a single-allocation store
    if (right->owned.size() == 1) { J->side_alloc[1] = right->owned[0]; J->side_bytes[1] = (size_t)right->device_bytes; }
    J->owned = left->owned;
    J->owned.insert(J->owned.end(), right->owned.begin(), right->owned.end());
    J->nvalues_dev = left->nvalues_dev + right->nvalues_dev;
    J->device_bytes = left->device_bytes + right->device_bytes;
    left->owned.clear(); right->owned.clear();
    left->d_values = right->d_values = nullptr;
    dmrg_ops_free(left);
    dmrg_ops_free(right);
    *out = J;
    return DMRG_OK;
}

// Shared core of dmrg_ops_add_lincombs / dmrg_ops_derive: forms the blocks of `n_lin_ops` linear combinations of operators of `S`
// in a fresh device allocation (*d_new_out) and returns their tables with offsets relative to that allocation.
static int form_lincombs(const dmrg_ops* S, const dmrg_op_desc* lin_ops, int32_t n_lin_ops, const int64_t* lin_ptr, const int32_t* lin_op,
                         const double* lin_coef, const int32_t* lin_trans, int32_t nlin, const char* who, double** d_new_out, int64_t* top_out,
                         std::vector<std::vector<int64_t>>& new_off, std::vector<std::vector<int32_t>>& new_colsec) {
    const int nops0 = (int)S->ops.size();
    std::vector<LinDesc2> lind;
    std::vector<LinSummand2> lins;
    int64_t top = 0;
    for (int q = 0; q < n_lin_ops; q++) {
        const dmrg_op_desc& d = lin_ops[q];
        DMRG_REQUIRE((d.side == 0 || d.side == 1) && d.p >= 0 && d.p < nlin, "%s: op %d: bad side or lin_ptr row", who, q);
        const auto& sec = S->sec[d.side];
        const int ns = (int)sec.size();
        const int64_t i0 = lin_ptr[d.p], i1 = lin_ptr[d.p + 1];
        DMRG_REQUIRE(i0 <= i1, "%s: lin_ptr not monotone", who);
        for (int64_t i = i0; i < i1; i++) {
            const int s = lin_op[i];
            const int sg = (lin_trans && lin_trans[i]) ? -1 : 1;
            DMRG_REQUIRE(s >= 0 && s < nops0 && S->ops[s].side == d.side && sg * S->ops[s].dn == d.dn && sg * S->ops[s].d2sz == d.d2sz,
                         "%s: op %d: summand %d is not an operator of the same side and (signed) charge", who, q, s);
        }
        std::vector<int64_t> ro(ns, -1);
        std::vector<int32_t> cs(ns, -1);
        for (int r = 0; r < ns; r++) {
            const int c = cs[r] = find_sec(sec, sec[r].n - d.dn, sec[r].two_sz - d.d2sz);
            if (c < 0) continue;
            // summand block feeding dst block (r, c): normal: the summand's block in row sector r; transposed: its block in row sector c
            // (whose column sector is then r)
            auto src_of = [&](int64_t i) -> int64_t { return (lin_trans && lin_trans[i]) ? S->row_off[lin_op[i]][c] : S->row_off[lin_op[i]][r]; };
            bool any = false;
            for (int64_t i = i0; i < i1; i++) any = any || src_of(i) >= 0;
            if (!any) continue;
            const int ld = (int)round_up2(sec[c].dim);
            LinDesc2 ld2{top, sec[r].dim, sec[c].dim, ld, 0, (int32_t)lins.size(), 0};
            for (int64_t i = i0; i < i1; i++) {
                const int64_t so = src_of(i);
                const int tr = (lin_trans && lin_trans[i]) ? 1 : 0;
                lins.push_back({so >= 0 ? so : 0, lin_coef[i], so >= 0 ? 1 : 0, tr, (int32_t)round_up2(tr ? sec[r].dim : sec[c].dim), 0});
            }
            ld2.sum_end = (int32_t)lins.size();
            lind.push_back(ld2);
            ro[r] = top;
            top += (int64_t)sec[r].dim * ld;
        }
        new_off.push_back(std::move(ro));
        new_colsec.push_back(std::move(cs));
    }
    double* d_new = nullptr;
    DMRG_CUDA(cudaMalloc(&d_new, sizeof(double) * (size_t)std::max<int64_t>(top, 2)));
    const int64_t delta = (int64_t)(d_new - S->d_values);   // the kernel addresses everything relative to S->d_values (signed offsets)
    for (auto& l : lind) l.dst += delta;
    int rc = DMRG_OK;
    if (!lind.empty()) {
        LinDesc2* d_lind = nullptr;
        LinSummand2* d_lins = nullptr;
        cudaError_t e = cudaMalloc(&d_lind, sizeof(LinDesc2) * lind.size());
        if (e == cudaSuccess) e = cudaMalloc(&d_lins, sizeof(LinSummand2) * lins.size());
        if (e == cudaSuccess) e = cudaMemcpy(d_lind, lind.data(), sizeof(LinDesc2) * lind.size(), cudaMemcpyHostToDevice);
        if (e == cudaSuccess) e = cudaMemcpy(d_lins, lins.data(), sizeof(LinSummand2) * lins.size(), cudaMemcpyHostToDevice);
        for (size_t y0 = 0; e == cudaSuccess && y0 < lind.size(); y0 += 32768) {
            const unsigned ny = (unsigned)std::min<size_t>(32768, lind.size() - y0);
            lincomb2_kernel<<<dim3(8, ny), 256>>>(d_lind + y0, d_lins, S->d_values);
            e = cudaGetLastError();
        }
        if (e == cudaSuccess) e = cudaDeviceSynchronize();
        cudaFree(d_lind);
        cudaFree(d_lins);
        if (e != cudaSuccess) { set_error("%s: %s", who, cudaGetErrorString(e)); rc = DMRG_ECUDA; }
    }
    if (rc != DMRG_OK) { cudaFree(d_new); return rc; }
    *d_new_out = d_new;
    *top_out = top;
    return DMRG_OK;
}

int dmrg_ops_add_lincombs(dmrg_ops* S, const dmrg_op_desc* lin_ops, int32_t n_lin_ops, const int64_t* lin_ptr, const int32_t* lin_op,
                          const double* lin_coef, const int32_t* lin_trans, int32_t nlin) {
    if (!S || !lin_ops || n_lin_ops <= 0 || !lin_ptr || !lin_op || !lin_coef) { set_error("dmrg_ops_add_lincombs: NULL or empty argument"); return DMRG_EINVAL; }
    if (S->cplx) { set_error("%s: complex stores (dmrg_ops_load_z) are served by dmrg_plan_create_z / dmrg_sigma / dmrg_hdiag / dmrg_davidson only", "dmrg_ops_add_lincombs"); return DMRG_EINVAL; }
    if (S->structure_only || S->owned.empty() || S->r_released) { set_error("dmrg_ops_add_lincombs: the store holds no device values (or its R side was released)"); return DMRG_EINVAL; }
    std::vector<std::vector<int64_t>> new_off;
    std::vector<std::vector<int32_t>> new_colsec;
    double* d_new = nullptr;
    int64_t top = 0;
    int rc;
    try {
        rc = form_lincombs(S, lin_ops, n_lin_ops, lin_ptr, lin_op, lin_coef, lin_trans, nlin, "dmrg_ops_add_lincombs", &d_new, &top, new_off, new_colsec);
    } catch (const std::bad_alloc&) { set_error("dmrg_ops_add_lincombs: out of host memory"); rc = DMRG_ENOMEM; }
    if (rc != DMRG_OK) return rc;
    if (d_new < S->d_values) rebase(S, d_new);   // keep every offset of the store >= 0 (< 0 means "absent" / "identity")
    const int64_t delta = (int64_t)(d_new - S->d_values);
    S->owned.push_back(d_new);
    for (int q = 0; q < n_lin_ops; q++) {
        dmrg_op_desc d = lin_ops[q];
        d.kind = DMRG_OP_LINCOMB; d.first_block = 0; d.nblocks = 0;
        S->ops.push_back(d);
        for (auto& o : new_off[q]) if (o >= 0) o += delta;
        S->row_off.push_back(std::move(new_off[q]));
        S->colsec.push_back(std::move(new_colsec[q]));
    }
    S->nvalues_dev += top;
    S->device_bytes += sizeof(double) * (size_t)std::max<int64_t>(top, 2);
    return DMRG_OK;
}

int dmrg_ops_derive(const dmrg_ops* src, const dmrg_op_desc* lin_ops, int32_t n_lin_ops, const int64_t* lin_ptr, const int32_t* lin_op,
                    const double* lin_coef, const int32_t* lin_trans, int32_t nlin, dmrg_ops** out) {
    if (!out) { set_error("dmrg_ops_derive: out is NULL"); return DMRG_EINVAL; }
    *out = nullptr;
    if (!src || !lin_ops || n_lin_ops <= 0 || !lin_ptr || !lin_op || !lin_coef) { set_error("dmrg_ops_derive: NULL or empty argument"); return DMRG_EINVAL; }
    if (src->cplx) { set_error("%s: complex stores (dmrg_ops_load_z) are served by dmrg_plan_create_z / dmrg_sigma / dmrg_hdiag / dmrg_davidson only", "dmrg_ops_derive"); return DMRG_EINVAL; }
    if (src->structure_only || src->owned.empty() || src->r_released) { set_error("dmrg_ops_derive: the source store holds no device values (or its R side was released)"); return DMRG_EINVAL; }
    dmrg_ops* D = new (std::nothrow) dmrg_ops();
    if (!D) { set_error("dmrg_ops_derive: out of host memory"); return DMRG_ENOMEM; }
    double* d_new = nullptr;
    int64_t top = 0;
    int rc;
    try {
        rc = form_lincombs(src, lin_ops, n_lin_ops, lin_ptr, lin_op, lin_coef, lin_trans, nlin, "dmrg_ops_derive", &d_new, &top, D->row_off, D->colsec);
    } catch (const std::bad_alloc&) { set_error("dmrg_ops_derive: out of host memory"); rc = DMRG_ENOMEM; }
    if (rc != DMRG_OK) { delete D; return rc; }
    D->sec[0] = src->sec[0];
    D->sec[1] = src->sec[1];
    for (int q = 0; q < n_lin_ops; q++) {
        dmrg_op_desc d = lin_ops[q];
        d.first_block = 0; d.nblocks = 0;
        D->ops.push_back(d);   // kind, p, q as the caller labels them: in the new store these are stored operators
    }
    D->d_values = d_new;
    D->owned.push_back(d_new);
    D->nvalues_dev = top;
    D->device_bytes = sizeof(double) * (size_t)std::max<int64_t>(top, 2);
    *out = D;
    return DMRG_OK;
}

}  // extern "C"
