// Internal definitions shared by the translation units of libdmrg_sigma.so (not part of the ABI).
#pragma once
#include <cuda_runtime.h>
#include <cstdarg>
#include <cstdint>
#include <cstdio>
#include <algorithm>
#include <string>
#include <thread>
#include <vector>

#include "../../include/dmrg_sigma.h"

namespace dmrg {

void set_error(const char* fmt, ...);

#define DMRG_CUDA(call)                                                                          \
    do {                                                                                         \
        cudaError_t e_ = (call);                                                                 \
        if (e_ != cudaSuccess) {                                                                 \
            dmrg::set_error("%s:%d: %s -> %s", __FILE__, __LINE__, #call, cudaGetErrorString(e_)); \
            return (e_ == cudaErrorMemoryAllocation) ? DMRG_ENOMEM : DMRG_ECUDA;                 \
        }                                                                                        \
    } while (0)

#define DMRG_REQUIRE(cond, ...)               \
    do {                                      \
        if (!(cond)) {                        \
            dmrg::set_error(__VA_ARGS__);     \
            return DMRG_EINVAL;               \
        }                                     \
    } while (0)

static inline int64_t round_up2(int64_t x) { return (x + 1) & ~int64_t(1); }

// ---- address spaces of GEMM operands -------------------------------------------------------
enum Space : uint32_t { SP_OPS = 0, SP_X = 1, SP_PSI = 2, SP_SIGMA = 3 };

// Segment flags
enum : uint32_t {
    SEG_A_MCONTIG = 1u << 0,   // A(m,k) at a_off + k*lda + m   (operator block used transposed)
    SEG_B_KCONTIG = 1u << 1,   // B(k,n) at b_off + n*ldb + k   (X = psi * O^T with O stored [n][k])
    SEG_A_IDENT   = 1u << 2,   // A is the identity: acc += alpha * B tile (no GEMM)
    // (bits 3, 4 unused: every operand the planner emits is 16-byte aligned with an even leading dimension)
    SEG_ALPHA_ONE = 1u << 5,   // alpha == +1 (set by the planner before upload)
    SEG_ALPHA_NEG = 1u << 6,   // alpha == -1
    SEG_A_SPACE_SHIFT = 8,     // 2 bits
    SEG_B_SPACE_SHIFT = 10,    // 2 bits
};

// One K-segment of a grouped GEMM job:  C += alpha * A(M x K) * B(K x N)
// Operands are addressed twice: as (space, offset, ld) for the cp.async path and the identity-A prologue, and as a
// tensor map for the TMA path.  A tensor map covers exactly the operand (an operator block, an X slice, a psi
// block, a packed R stack), so everything outside it is zero-filled by the TMA unit; the one exception is the
// stage-1 A operand, a run of psi rows inside its panel's map, whose first row is a_o0.  The TMA box of a map is
// sized to the operand (planner: box_shape): a_pitch / b_pitch = its inner dimension in doubles = the row pitch of
// the shared-memory tile (always = 4 mod 8: conflict-free fragment loads), a_bytes / b_bytes = its size.
struct Seg {
    int64_t  a_off;
    int64_t  b_off;
    int32_t  lda, ldb;
    int32_t  K;
    uint32_t flags;
    double   alpha;
    int32_t  a_map, b_map;
    int32_t  a_o0;
    uint16_t a_pitch, b_pitch;
    uint32_t a_bytes, b_bytes;
};
static_assert(sizeof(Seg) == 64, "Seg layout");

// 128-byte CUtensorMap image (cuda.h is not included here; the planner encodes it through the driver entry point)
struct alignas(64) TensorMap { uint64_t opaque[16]; };
enum : int { COPY_LDGSTS = 1, COPY_TMA = 2 };

enum : uint32_t { JOB_BETA1 = 1u << 0, JOB_C_SPACE_SHIFT = 8 };

// One output matrix: C (M x N, row-major, ldc) = beta*C + sum over segments
struct Job {
    int64_t  c_off;
    int32_t  ldc, M, N;
    int32_t  seg_begin, seg_end;
    uint32_t flags;
    int32_t  nstages;   // pipeline stages of GEMM_BK k-columns over all non-identity segments (planner)
};
static_assert(sizeof(Job) == 40, "Job layout");

// One CTA of work: rows [m0, m0+rows) x cols [n0, n0+cols) of job; rows <= BM, cols <= BN of the kernel
// variant (the planner cuts a dimension into full pieces plus the remainder).
struct Tile {
    int32_t  job;
    int32_t  m0, n0;
    uint16_t rows, cols;   // rows: of the LAST sub-tile when the tile is a run of M sub-tiles (reps > 1); the others are full
    uint16_t reps = 1;     // consecutive BM-row sub-tiles this CTA computes one after the other (same columns)
    uint16_t pad_ = 0;
};
static_assert(sizeof(Tile) == 20, "Tile layout");

// What the kernel reads per CTA: the tile and everything it needs of its job in ONE 64-byte record, so that a CTA's first
// global round trip is its only descriptor fetch before the segment list (tile -> job -> first non-identity segment used
// to be three dependent loads, which short tiles -- a couple of pipeline stages -- cannot hide).  a_map0 / b_map0: the
// tensor maps of the first GEMM segment, prefetched while that segment's descriptor is still on its way.
struct alignas(64) TileDesc {
    int64_t  c_off;
    int32_t  ldc;
    int32_t  m0, n0;
    uint16_t rows, cols;
    int32_t  seg_begin, seg_gemm, seg_end;   // [seg_begin, seg_gemm): identity-A segments, [seg_gemm, seg_end): GEMM segments
    uint32_t flags;                          // JOB_*
    int32_t  nstages;
    int32_t  a_map0, b_map0;
    int32_t  reps;                           // M sub-tiles of the kernel's BM rows computed back to back by this CTA (rows = those of the last one)
    int32_t  pad_[2];
};
static_assert(sizeof(TileDesc) == 64, "TileDesc layout");

inline std::vector<TileDesc> make_tile_descs(const std::vector<Tile>& tiles, const std::vector<Job>& jobs, const std::vector<Seg>& segs) {
    std::vector<int32_t> first_gemm(jobs.size());
    std::vector<TileDesc> out(tiles.size());
    const unsigned nthr = std::max(1u, std::min(32u, std::thread::hardware_concurrency()));
    auto parallel_for = [&](size_t n, auto&& body) {   // body(begin, end) on contiguous slices, all host threads
        std::vector<std::thread> pool;
        const size_t per = (n + nthr - 1) / nthr;
        for (unsigned t = 1; t < nthr; t++)
            if (t * per < n) pool.emplace_back([&, t] { body(t * per, std::min(n, (t + 1) * per)); });
        body(0, std::min(n, per));
        for (auto& th : pool) th.join();
    };
    parallel_for(jobs.size(), [&](size_t lo, size_t hi) {
        for (size_t j = lo; j < hi; j++) {
            int32_t s = jobs[j].seg_begin;
            while (s < jobs[j].seg_end && (segs[s].flags & SEG_A_IDENT)) s++;
            first_gemm[j] = s;
        }
    });
    parallel_for(tiles.size(), [&](size_t lo, size_t hi) {
        for (size_t t = lo; t < hi; t++) {
            const Tile& T = tiles[t];
            const Job& J = jobs[T.job];
            TileDesc& d = out[t];
            d.c_off = J.c_off; d.ldc = J.ldc; d.m0 = T.m0; d.n0 = T.n0; d.rows = T.rows; d.cols = T.cols;
            d.seg_begin = J.seg_begin; d.seg_gemm = first_gemm[T.job]; d.seg_end = J.seg_end;
            d.flags = J.flags; d.nstages = J.nstages;
            const bool has = d.seg_gemm < d.seg_end;
            d.a_map0 = has ? segs[d.seg_gemm].a_map : 0; d.b_map0 = has ? segs[d.seg_gemm].b_map : 0;
            d.reps = T.reps;
            d.pad_[0] = d.pad_[1] = 0;
        }
    });
    return out;
}

// tile shape of the grouped GEMM kernel (one: 64 x 64); launch variant 0 = single tiles, 1 = tiles may be runs of M sub-tiles
struct TileShape { int bm, bn; };
constexpr int NUM_VARIANTS = 1;
extern const TileShape kVariants[NUM_VARIANTS];
#ifndef DMRG_GEMM_BK
#define DMRG_GEMM_BK 32
#endif
constexpr int GEMM_BK = DMRG_GEMM_BK;   // k-columns per pipeline stage (8, 16 or 32); 32 measured best at cfg 5 / cfg 3

int launch_grouped_gemm(int variant, int copy_mode, const Seg* segs, const TileDesc* tiles, int64_t ntiles,
                        const double* ops, double* xws, const double* psi, double* sigma, const TensorMap* tmaps, cudaStream_t st);
int gemm_init();   // sets shared-memory attributes once

}  // namespace dmrg

// ---- the operator store ---------------------------------------------------------------------
struct dmrg_ops {
    std::vector<dmrg_sector> sec[2];
    std::vector<dmrg_op_desc> ops;
    // per op, per ROW sector: device offset of the block (doubles) or -1; the column sector that the
    // charge implies (or -1); all blocks are row-major with leading dimension round_up2(dim[col]).
    std::vector<std::vector<int64_t>> row_off;
    std::vector<std::vector<int32_t>> colsec;
    double* d_values = nullptr;    // base of the store's address space: every block offset is relative to it
    std::vector<double*> owned;    // device allocations the store owns (d_values first; joined / appended arrays after it)
    double* side_alloc[2] = {nullptr, nullptr};   // dmrg_ops_load: the allocation holding the L-side / R-side blocks (also in `owned`)
    size_t side_bytes[2] = {0, 0};
    mutable bool r_released = false;   // a plan created with release_r_store freed side_alloc[1]: the store serves that plan only
    bool cplx = false;             // dmrg_ops_load_z: complex blocks (L side: real 2x2-image blocks, R side: row-planar re | im; ops_store.cu)
    bool structure_only = false;   // loaded with values == NULL: planning / statistics only, no device memory
    int64_t nvalues_dev = 0;     // doubles allocated (stored + lincomb, padded)
    int64_t device_bytes = 0;
};
