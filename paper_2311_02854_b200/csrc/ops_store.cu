// dmrg_ops_load: block-sparse operator store in HBM (Eq. 19-24; Fig. 1b) and the
// "intermediates" step O = sum_s alpha_s a_s, done once per bond at load time
// because it does not depend on psi.
//
// HBM layout: one flat FP64 array.  Block (op, row sector r) is a row-major dim[r] x dim[c] matrix
// whose rows are padded to an even leading dimension, so that every row starts 16-byte aligned and
// the GEMM kernels can stage it with 16-byte cp.async.
#include <algorithm>
#include <cstring>
#include <new>

#include "common.h"

namespace dmrg {

static thread_local std::string g_err;
void set_error(const char* fmt, ...) {
    char buf[1024];
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(buf, sizeof buf, fmt, ap);
    va_end(ap);
    g_err = buf;
}

struct RepackDesc { int64_t src, dst; int32_t rows, cols, ld, side; int32_t mode, pad_; };   // side: which of the store's two allocations dst lives in (host bookkeeping)
// mode 0: real block.  Complex stores (dmrg_ops_load_z; src = interleaved (re, im) pairs, offsets in doubles):
//   mode 1, L side: the real 2 rows x 2 cols image with interleaved rows and columns, [2r+a][2c+b] = (a == b ? re : (a ? im : -im)),
//           so that  image(A) image(B) = image(A B),  image(A)^T = image(A^H),  and a complex matrix-vector product
//           becomes a real one on vectors whose entries are (re, im) row pairs -- stage 2 reads these blocks as they are;
//   mode 2, R side: row-planar, row r = [re(r, 0..cols) | im(r, 0..cols)], each half padded to an even length (ld = 2 halves);
//           stage 1 reads the R side through the plan's packed copy, which builds its own real image from this.

// dst[r*ld + c] = c < cols ? src[r*cols + c] : 0      one CTA per block
__global__ void __launch_bounds__(256) repack_kernel(const RepackDesc* __restrict__ desc, const double* __restrict__ src_base,
                                                     int64_t src_shift, double* __restrict__ dst_base) {
    const RepackDesc d = desc[blockIdx.x];
    const double* src = src_base + (d.src - src_shift);
    double* dst = dst_base + d.dst;
    if (d.mode == 1) {   // ld = 2 cols
        const int64_t n = (int64_t)2 * d.rows * d.ld;
        for (int64_t e = threadIdx.x; e < n; e += blockDim.x) {
            const int rr = (int)(e / d.ld), cc = (int)(e - (int64_t)rr * d.ld);
            const int a = rr & 1, b = cc & 1;
            const double v = src[2 * ((int64_t)(rr >> 1) * d.cols + (cc >> 1)) + (a ^ b)];
            dst[e] = (a == 0 && b == 1) ? -v : v;
        }
        return;
    }
    if (d.mode == 2) {   // ld = 2 round_up2(cols)
        const int half = d.ld / 2;
        const int64_t n = (int64_t)d.rows * d.ld;
        for (int64_t e = threadIdx.x; e < n; e += blockDim.x) {
            const int r = (int)(e / d.ld), cc = (int)(e - (int64_t)r * d.ld);
            const int part = cc >= half, c = cc - part * half;
            dst[e] = c < d.cols ? src[2 * ((int64_t)r * d.cols + c) + part] : 0.0;
        }
        return;
    }
    const int64_t n = (int64_t)d.rows * d.ld;
    for (int64_t e = threadIdx.x; e < n; e += blockDim.x) {
        int r = (int)(e / d.ld), c = (int)(e - (int64_t)r * d.ld);
        dst[e] = c < d.cols ? src[(int64_t)r * d.cols + c] : 0.0;
    }
}

struct LinDesc { int64_t dst; int64_t n; int32_t sum_begin, sum_end; };
struct LinSummand { int64_t src; double coef; };   // src < 0: block absent in this summand

// dst[e] = sum_i coef_i * src_i[e]  in summand order (deterministic)      grid (chunks, lincomb blocks)
__global__ void __launch_bounds__(256) lincomb_kernel(const LinDesc* __restrict__ desc, const LinSummand* __restrict__ sums,
                                                      double* __restrict__ vals) {
    const LinDesc d = desc[blockIdx.y];
    for (int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; e < d.n; e += (int64_t)gridDim.x * blockDim.x) {
        double acc = 0.0;
        for (int i = d.sum_begin; i < d.sum_end; i++) {
            const LinSummand s = sums[i];
            if (s.src >= 0) acc = fma(s.coef, vals[s.src + e], acc);
        }
        vals[d.dst + e] = acc;
    }
}

// Complex stores: out = sum_i (cr_i + i ci_i) * src_i in summand order.  In both device layouts a complex entry is a pair of
// doubles (x, y) = (re, im) at positions (p, p + delta): the L-side image keeps them in rows 2r / 2r + 1 of one column
// (x = [2r][c] carries re for even c and -im for odd c, y = [2r+1][c] the matching im / re: multiplying by i maps
// (x, y) -> (-y, x) in every column), the R-side row-planar layout in the two halves of a row.  Pair q of a block sits at
// p = (q / w) * stride + q % w.
struct LinDescZ { int64_t dst; int64_t npairs; int32_t w, stride, delta; int32_t sum_begin, sum_end, pad_; };
struct LinSummandZ { int64_t src; double cr, ci; };
__global__ void __launch_bounds__(256) lincomb_z_kernel(const LinDescZ* __restrict__ desc, const LinSummandZ* __restrict__ sums,
                                                        double* __restrict__ vals) {
    const LinDescZ d = desc[blockIdx.y];
    for (int64_t q = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; q < d.npairs; q += (int64_t)gridDim.x * blockDim.x) {
        const int64_t p = (q / d.w) * d.stride + q % d.w;
        double ax = 0.0, ay = 0.0;
        for (int i = d.sum_begin; i < d.sum_end; i++) {
            const LinSummandZ s = sums[i];
            if (s.src < 0) continue;
            const double x = vals[s.src + p], y = vals[s.src + p + d.delta];
            ax += s.cr * x - s.ci * y;
            ay += s.cr * y + s.ci * x;
        }
        vals[d.dst + p] = ax;
        vals[d.dst + p + d.delta] = ay;
    }
}

static int find_sector(const std::vector<dmrg_sector>& s, int n, int two_sz) {
    for (size_t i = 0; i < s.size(); i++)
        if (s[i].n == n && s[i].two_sz == two_sz) return (int)i;
    return -1;
}

static int ops_load_impl(const dmrg_sector* secL, int32_t nsecL, const dmrg_sector* secR, int32_t nsecR,
                         const dmrg_op_desc* ops, int32_t nops, const dmrg_block_desc* blocks, int64_t nblocks,
                         const double* values, int64_t nvalues, int32_t values_on_device,
                         const int64_t* lin_ptr, const int32_t* lin_op, const double* lin_coef, int32_t nlin,
                         bool cplx, dmrg_ops* S) {
    S->cplx = cplx;   // values / lin_coef are interleaved (re, im) pairs; nvalues and block offsets count complex numbers
    DMRG_REQUIRE((secL || nsecL == 0) && (secR || nsecR == 0) && nsecL >= 0 && nsecR >= 0 && nsecL + nsecR > 0, "dmrg_ops_load: empty sector table");
    DMRG_REQUIRE(nops >= 0 && nblocks >= 0 && nvalues >= 0, "dmrg_ops_load: negative count");
    DMRG_REQUIRE(nops == 0 || ops, "dmrg_ops_load: ops is NULL");
    DMRG_REQUIRE(nblocks == 0 || blocks, "dmrg_ops_load: blocks is NULL");
    S->structure_only = (values == nullptr);
    DMRG_REQUIRE(nlin == 0 || (lin_ptr && lin_op && lin_coef), "dmrg_ops_load: lincomb arrays are NULL");
    if (!S->structure_only) {
        int ndev = 0;
        DMRG_CUDA(cudaGetDeviceCount(&ndev));
    }
    if (nsecL) S->sec[0].assign(secL, secL + nsecL);
    if (nsecR) S->sec[1].assign(secR, secR + nsecR);
    for (int side = 0; side < 2; side++)
        for (auto& s : S->sec[side]) DMRG_REQUIRE(s.dim > 0, "dmrg_ops_load: sector with dim <= 0");
    S->ops.assign(ops, ops + nops);
    S->row_off.resize(nops);
    S->colsec.resize(nops);

    std::vector<RepackDesc> rep;
    rep.reserve(nblocks);
    // L-side and R-side blocks live in two device allocations (the R side can be released once a plan has packed it,
    // dmrg_plan_options.release_r_store); while the layout is computed, offsets are local to their side's allocation
    int64_t tops[2] = {0, 0};   // device doubles per side
    for (int o = 0; o < nops; o++) {
        const dmrg_op_desc& d = ops[o];
        DMRG_REQUIRE(d.side == 0 || d.side == 1, "dmrg_ops_load: op %d has side %d", o, d.side);
        const auto& sec = S->sec[d.side];
        const int ns = (int)sec.size();
        S->row_off[o].assign(ns, -1);
        S->colsec[o].assign(ns, -1);
        for (int r = 0; r < ns; r++) S->colsec[o][r] = find_sector(sec, sec[r].n - d.dn, sec[r].two_sz - d.d2sz);
        if (d.kind == DMRG_OP_LINCOMB) continue;
        DMRG_REQUIRE(d.nblocks >= 0 && d.first_block >= 0 && d.first_block + d.nblocks <= nblocks,
                     "dmrg_ops_load: op %d block range out of bounds", o);
        for (int64_t b = d.first_block; b < d.first_block + d.nblocks; b++) {
            const dmrg_block_desc& bd = blocks[b];
            DMRG_REQUIRE(bd.row_sector >= 0 && bd.row_sector < ns && bd.col_sector >= 0 && bd.col_sector < ns,
                         "dmrg_ops_load: block %lld sector index out of range", (long long)b);
            DMRG_REQUIRE(S->colsec[o][bd.row_sector] == bd.col_sector,
                         "dmrg_ops_load: block %lld of op %d violates the operator charge", (long long)b, o);
            DMRG_REQUIRE(S->row_off[o][bd.row_sector] < 0, "dmrg_ops_load: op %d has two blocks in row sector %d", o,
                         bd.row_sector);
            const int rows = sec[bd.row_sector].dim, cols = sec[bd.col_sector].dim;
            DMRG_REQUIRE(bd.offset >= 0 && bd.offset + (int64_t)rows * cols <= nvalues,
                         "dmrg_ops_load: block %lld exceeds values[]", (long long)b);
            int64_t& top = tops[d.side];
            S->row_off[o][bd.row_sector] = top;
            if (!cplx) {
                const int ld = (int)round_up2(cols);
                rep.push_back({bd.offset, top, rows, cols, ld, d.side, 0, 0});
                top += (int64_t)rows * ld;
            } else if (d.side == 0) {
                rep.push_back({2 * bd.offset, top, rows, cols, 2 * cols, d.side, 1, 0});
                top += (int64_t)4 * rows * cols;
            } else {
                const int ld = 2 * (int)round_up2(cols);
                rep.push_back({2 * bd.offset, top, rows, cols, ld, d.side, 2, 0});
                top += (int64_t)rows * ld;
            }
        }
    }
    // linear combinations: block present where any summand has one
    std::vector<LinDesc> lind;
    std::vector<LinSummand> lins;
    std::vector<LinDescZ> lindz;
    std::vector<LinSummandZ> linsz;
    std::vector<int> lin_side;   // side of lind[i] (its summands are on the same side)
    for (int o = 0; o < nops; o++) {
        const dmrg_op_desc& d = ops[o];
        if (d.kind != DMRG_OP_LINCOMB) continue;
        DMRG_REQUIRE(d.p >= 0 && d.p < nlin, "dmrg_ops_load: LINCOMB op %d refers to row %d of lin_ptr (nlin=%d)", o, d.p, nlin);
        const auto& sec = S->sec[d.side];
        const int ns = (int)sec.size();
        const int64_t i0 = lin_ptr[d.p], i1 = lin_ptr[d.p + 1];
        DMRG_REQUIRE(i0 <= i1, "dmrg_ops_load: lin_ptr not monotone");
        for (int64_t i = i0; i < i1; i++) {
            const int s = lin_op[i];
            DMRG_REQUIRE(s >= 0 && s < nops && ops[s].kind != DMRG_OP_LINCOMB && ops[s].side == d.side &&
                             ops[s].dn == d.dn && ops[s].d2sz == d.d2sz,
                         "dmrg_ops_load: LINCOMB op %d: summand %d is not a stored operator of the same side and charge", o, s);
        }
        for (int r = 0; r < ns; r++) {
            const int c = S->colsec[o][r];
            if (c < 0) continue;
            bool any = false;
            for (int64_t i = i0; i < i1; i++) any = any || S->row_off[lin_op[i]][r] >= 0;
            if (!any) continue;
            int64_t& top = tops[d.side];
            if (cplx) {
                const int rows = sec[r].dim, cols = sec[c].dim, pc = (int)round_up2(cols);
                LinDescZ ld = d.side == 0 ? LinDescZ{top, (int64_t)rows * 2 * cols, 2 * cols, 4 * cols, 2 * cols, (int32_t)linsz.size(), 0, 0}
                                          : LinDescZ{top, (int64_t)rows * pc, pc, 2 * pc, pc, (int32_t)linsz.size(), 0, 0};
                lin_side.push_back(d.side);
                for (int64_t i = i0; i < i1; i++) linsz.push_back({S->row_off[lin_op[i]][r], lin_coef[2 * i], lin_coef[2 * i + 1]});
                ld.sum_end = (int32_t)linsz.size();
                lindz.push_back(ld);
                S->row_off[o][r] = top;
                top += d.side == 0 ? (int64_t)4 * rows * cols : (int64_t)rows * 2 * pc;
                continue;
            }
            const int64_t n = (int64_t)sec[r].dim * round_up2(sec[c].dim);
            LinDesc ld{top, n, (int32_t)lins.size(), 0};
            lin_side.push_back(d.side);
            for (int64_t i = i0; i < i1; i++) lins.push_back({S->row_off[lin_op[i]][r], lin_coef[i]});
            ld.sum_end = (int32_t)lins.size();
            lind.push_back(ld);
            S->row_off[o][r] = top;
            top += n;
        }
    }
    S->nvalues_dev = tops[0] + tops[1];
    S->side_bytes[0] = tops[0] > 0 ? sizeof(double) * (size_t)std::max<int64_t>(tops[0], 2) : 0;
    S->side_bytes[1] = tops[1] > 0 ? sizeof(double) * (size_t)std::max<int64_t>(tops[1], 2) : 0;
    S->device_bytes = (int64_t)(S->side_bytes[0] + S->side_bytes[1]);
    if (S->structure_only) {   // planning only: one linear numbering, R behind L
        for (int o = 0; o < nops; o++)
            if (ops[o].side == 1)
                for (auto& off : S->row_off[o]) if (off >= 0) off += tops[0];
        return DMRG_OK;
    }
    double* side_ptr[2] = {nullptr, nullptr};
    for (int sd = 0; sd < 2; sd++)
        if (S->side_bytes[sd]) {
            DMRG_CUDA(cudaMalloc(&side_ptr[sd], S->side_bytes[sd]));
            S->owned.push_back(side_ptr[sd]);
            S->side_alloc[sd] = side_ptr[sd];
        }
    // one address space for both: offsets relative to the lower allocation (>= 0; both are cudaMalloc'ed, so the
    // distance is a multiple of 32 doubles and every row keeps its 16-byte alignment)
    S->d_values = side_ptr[0] && side_ptr[1] ? std::min(side_ptr[0], side_ptr[1]) : (side_ptr[0] ? side_ptr[0] : side_ptr[1]);
    DMRG_REQUIRE(S->d_values != nullptr, "dmrg_ops_load: the store has no blocks");
    const int64_t shift[2] = {side_ptr[0] ? (int64_t)(side_ptr[0] - S->d_values) : 0, side_ptr[1] ? (int64_t)(side_ptr[1] - S->d_values) : 0};
    for (int o = 0; o < nops; o++)
        for (auto& off : S->row_off[o]) if (off >= 0) off += shift[ops[o].side];
    for (auto& r : rep) r.dst += shift[r.side];
    for (size_t i = 0; i < lind.size(); i++) {
        lind[i].dst += shift[lin_side[i]];
        for (int q = lind[i].sum_begin; q < lind[i].sum_end; q++) if (lins[q].src >= 0) lins[q].src += shift[lin_side[i]];
    }
    for (size_t i = 0; i < lindz.size(); i++) {
        lindz[i].dst += shift[lin_side[i]];
        for (int q = lindz[i].sum_begin; q < lindz[i].sum_end; q++) if (linsz[q].src >= 0) linsz[q].src += shift[lin_side[i]];
    }

    // ---- repack stored blocks (row padding) -------------------------------------------------
    if (!rep.empty()) {
        std::sort(rep.begin(), rep.end(), [](const RepackDesc& a, const RepackDesc& b) { return a.src < b.src; });
        const int64_t CHUNK = int64_t(1) << 26;   // 64 Mi doubles = 512 MiB staging
        const int64_t esz = cplx ? 2 : 1;         // doubles per stored number; RepackDesc.src counts doubles
        const int64_t nvalues_d = nvalues * esz;
        auto raw_end = [&](const RepackDesc& r) { return r.src + esz * (int64_t)r.rows * r.cols; };
        double* d_stage = nullptr;
        RepackDesc* d_desc = nullptr;
        const size_t DESC_BATCH = 1 << 16;
        DMRG_CUDA(cudaMalloc(&d_desc, sizeof(RepackDesc) * DESC_BATCH));
        int64_t stage_cap = 0;
        size_t i = 0;
        int rc = DMRG_OK;
        while (i < rep.size() && rc == DMRG_OK) {
            // batch [i, j): raw extent <= CHUNK (or a single oversized block), at most DESC_BATCH blocks
            const int64_t lo = rep[i].src;
            int64_t hi = lo;
            size_t j = i;
            while (j < rep.size() && j - i < DESC_BATCH) {
                const int64_t end = raw_end(rep[j]);
                if (j > i && end - lo > CHUNK) break;
                hi = std::max(hi, end);
                j++;
            }
            const double* src_base = nullptr;
            if (values_on_device) {
                src_base = values + lo;
            } else {
                if (hi - lo > stage_cap) {
                    if (d_stage) cudaFree(d_stage);
                    d_stage = nullptr;
                    stage_cap = std::max(hi - lo, std::min<int64_t>(CHUNK, nvalues_d));
                    cudaError_t e = cudaMalloc(&d_stage, sizeof(double) * (size_t)stage_cap);
                    if (e != cudaSuccess) { set_error("dmrg_ops_load: staging cudaMalloc failed"); rc = DMRG_ENOMEM; break; }
                }
                cudaError_t e = cudaMemcpy(d_stage, values + lo, sizeof(double) * (size_t)(hi - lo), cudaMemcpyHostToDevice);
                if (e != cudaSuccess) { set_error("dmrg_ops_load: H2D copy failed: %s", cudaGetErrorString(e)); rc = DMRG_ECUDA; break; }
                src_base = d_stage;
            }
            cudaError_t e = cudaMemcpy(d_desc, rep.data() + i, sizeof(RepackDesc) * (j - i), cudaMemcpyHostToDevice);
            if (e == cudaSuccess) {
                repack_kernel<<<(unsigned)(j - i), 256>>>(d_desc, src_base, lo, S->d_values);
                e = cudaDeviceSynchronize();
            }
            if (e != cudaSuccess) { set_error("dmrg_ops_load: repack failed: %s", cudaGetErrorString(e)); rc = DMRG_ECUDA; break; }
            i = j;
        }
        if (d_stage) cudaFree(d_stage);
        cudaFree(d_desc);
        if (rc != DMRG_OK) return rc;
    }
    // ---- intermediates: O = sum_s alpha_s a_s, block by block ------------------
    if (!lindz.empty()) {
        LinDescZ* d_lind = nullptr;
        LinSummandZ* d_lins = nullptr;
        DMRG_CUDA(cudaMalloc(&d_lind, sizeof(LinDescZ) * lindz.size()));
        DMRG_CUDA(cudaMalloc(&d_lins, sizeof(LinSummandZ) * linsz.size()));
        DMRG_CUDA(cudaMemcpy(d_lind, lindz.data(), sizeof(LinDescZ) * lindz.size(), cudaMemcpyHostToDevice));
        DMRG_CUDA(cudaMemcpy(d_lins, linsz.data(), sizeof(LinSummandZ) * linsz.size(), cudaMemcpyHostToDevice));
        const size_t YB = 32768;
        for (size_t y0 = 0; y0 < lindz.size(); y0 += YB) {
            const unsigned ny = (unsigned)std::min(YB, lindz.size() - y0);
            lincomb_z_kernel<<<dim3(8, ny), 256>>>(d_lind + y0, d_lins, S->d_values);
        }
        DMRG_CUDA(cudaGetLastError());
        DMRG_CUDA(cudaDeviceSynchronize());
        cudaFree(d_lind);
        cudaFree(d_lins);
    }
    if (!lind.empty()) {
        LinDesc* d_lind = nullptr;
        LinSummand* d_lins = nullptr;
        DMRG_CUDA(cudaMalloc(&d_lind, sizeof(LinDesc) * lind.size()));
        DMRG_CUDA(cudaMalloc(&d_lins, sizeof(LinSummand) * lins.size()));
        DMRG_CUDA(cudaMemcpy(d_lind, lind.data(), sizeof(LinDesc) * lind.size(), cudaMemcpyHostToDevice));
        DMRG_CUDA(cudaMemcpy(d_lins, lins.data(), sizeof(LinSummand) * lins.size(), cudaMemcpyHostToDevice));
        const size_t YB = 32768;
        for (size_t y0 = 0; y0 < lind.size(); y0 += YB) {
            const unsigned ny = (unsigned)std::min(YB, lind.size() - y0);
            lincomb_kernel<<<dim3(8, ny), 256>>>(d_lind + y0, d_lins, S->d_values);
        }
        DMRG_CUDA(cudaGetLastError());
        DMRG_CUDA(cudaDeviceSynchronize());
        cudaFree(d_lind);
        cudaFree(d_lins);
    }
    return DMRG_OK;
}

}  // namespace dmrg

extern "C" {

int dmrg_ops_load(const dmrg_sector* secL, int32_t nsecL, const dmrg_sector* secR, int32_t nsecR,
                  const dmrg_op_desc* ops, int32_t nops, const dmrg_block_desc* blocks, int64_t nblocks,
                  const double* values, int64_t nvalues, int32_t values_on_device,
                  const int64_t* lin_ptr, const int32_t* lin_op, const double* lin_coef, int32_t nlin,
                  dmrg_ops** out) {
    if (!out) { dmrg::set_error("dmrg_ops_load: out is NULL"); return DMRG_EINVAL; }
    *out = nullptr;
    dmrg_ops* S = new (std::nothrow) dmrg_ops();
    if (!S) { dmrg::set_error("dmrg_ops_load: out of host memory"); return DMRG_ENOMEM; }
    int rc;
    try {
        rc = dmrg::ops_load_impl(secL, nsecL, secR, nsecR, ops, nops, blocks, nblocks, values, nvalues, values_on_device,
                                 lin_ptr, lin_op, lin_coef, nlin, false, S);
    } catch (const std::bad_alloc&) {
        dmrg::set_error("dmrg_ops_load: out of host memory");
        rc = DMRG_ENOMEM;
    } catch (...) {
        dmrg::set_error("dmrg_ops_load: unexpected exception");
        rc = DMRG_EINVAL;
    }
    if (rc != DMRG_OK) { dmrg_ops_free(S); return rc; }
    *out = S;
    return DMRG_OK;
}

int dmrg_ops_load_z(const dmrg_sector* secL, int32_t nsecL, const dmrg_sector* secR, int32_t nsecR,
                    const dmrg_op_desc* ops, int32_t nops, const dmrg_block_desc* blocks, int64_t nblocks,
                    const double* values, int64_t nvalues, int32_t values_on_device,
                    const int64_t* lin_ptr, const int32_t* lin_op, const double* lin_coef, int32_t nlin,
                    dmrg_ops** out) {
    if (!out) { dmrg::set_error("dmrg_ops_load_z: out is NULL"); return DMRG_EINVAL; }
    *out = nullptr;
    dmrg_ops* S = new (std::nothrow) dmrg_ops();
    if (!S) { dmrg::set_error("dmrg_ops_load_z: out of host memory"); return DMRG_ENOMEM; }
    int rc;
    try {
        rc = dmrg::ops_load_impl(secL, nsecL, secR, nsecR, ops, nops, blocks, nblocks, values, nvalues, values_on_device,
                                 lin_ptr, lin_op, lin_coef, nlin, true, S);
    } catch (const std::bad_alloc&) {
        dmrg::set_error("dmrg_ops_load_z: out of host memory");
        rc = DMRG_ENOMEM;
    } catch (...) {
        dmrg::set_error("dmrg_ops_load_z: unexpected exception");
        rc = DMRG_EINVAL;
    }
    if (rc != DMRG_OK) { dmrg_ops_free(S); return rc; }
    *out = S;
    return DMRG_OK;
}

int32_t dmrg_ops_is_complex(const dmrg_ops* ops) { return ops && ops->cplx ? 1 : 0; }

void dmrg_ops_free(dmrg_ops* ops) {
    if (!ops) return;
    for (double* p : ops->owned) cudaFree(p);
    delete ops;
}

int64_t dmrg_ops_device_bytes(const dmrg_ops* ops) { return ops ? ops->device_bytes : 0; }

const char* dmrg_last_error(void) { return dmrg::g_err.c_str(); }
const char* dmrg_version(void) { return "dmrg_sigma_b200 0.1 (sm_100a, FP64 DMMA)"; }

}  // extern "C"
