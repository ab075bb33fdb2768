// dmrg_plan internals (not part of the ABI).
#pragma once
#include "common.h"

constexpr int64_t kHdIdent = INT64_MIN;   // HdItem offset of an identity factor (a packed R block can sit below the store: plain negatives are addresses)
struct HdItem { int64_t l_off, r_off; int32_t ldl, ldr; double alpha; int64_t l_im, r_im; int32_t part = 0, pad_ = 0; };   // l_im, r_im, part: complex plans (distance from the real to the imaginary part of a diagonal entry; 1 = imaginary-coefficient task)
struct HdTile { int32_t blk; int16_t ti, tj; };   // 32 x 32 tile of a psi block
struct HdBlock { int64_t offset; int32_t dl, dr; int32_t item_begin, item_end; int64_t pad_off; };   // pad_off: block in the padded psi copy

struct RedJob { int64_t sigma_off, part_off, part_stride; int32_t M, N, ldp, nparts; };   // split-K reduction of one sigma block

struct PackDesc { int64_t src, dst; int32_t dRo, dRi, src_ld, trans, ldp, pad_; int64_t im_delta; };   // im_delta (complex plans): from a block's real-part rows to its imaginary-part rows in the pack   // one R block copied into the packed stage-1 store

struct PlanLaunch { int variant; int stage; int64_t tile_begin, ntiles; };
struct PlanGroup { int stage; int first_launch, nlaunch; };   // launches of one stage of one chunk: mutually independent (stage 3: range of the RedJob table)

enum {
    ST_TASKS = 0, ST_ALG_FLOPS, ST_S1_FLOPS, ST_S2_FLOPS, ST_PADDED_FLOPS, ST_S1_JOBS, ST_CHUNKS, ST_LAUNCHES,
    ST_DEVICE_BYTES, ST_ALG_BYTES, ST_S1_TILES, ST_S2_TILES, ST_CANON_FLOPS, ST_STAGE_FLOPS, ST_TILE_FLOPS, ST_WARP_FLOPS, ST_XWS_ELEMS, ST_TENSOR_MAPS, ST_S1_FILL, ST_S2_FILL, ST_S1_STAGES, ST_S2_STAGES, ST_COUNT
};

struct DavidsonWs;
struct dmrg_comm;

struct dmrg_plan {
    const dmrg_ops* ops = nullptr;
    std::vector<dmrg_psi_block> blocks;
    std::vector<int64_t> shard_terms;   // indices (into the caller's term array) of the terms this plan evaluates, in plan order
    int64_t psi_size = 0;   // doubles in psi / sigma (2 per number for a complex plan)
    bool cplx = false;      // complex plan (dmrg_plan_create_z)
    double* d_sigz = nullptr;   // complex plan: the two row-planar accumulators of dmrg_sigma (2 * psi_size doubles)
    dmrg::Seg* d_segs = nullptr;
    dmrg::TileDesc* d_tiles = nullptr;   // one 64-byte record per CTA: the tile and its job (common.h)
    double* d_xws = nullptr;
    int64_t xws_elems = 0;
    std::vector<PlanLaunch> launches;
    std::vector<PlanGroup> groups;
    int copy_mode = 2;   // operand staging of the GEMM kernel (dmrg_plan_options.copy_mode)
    RedJob* d_reds = nullptr;
    double* d_psi_pad = nullptr;   // psi re-laid with even leading dimensions (16-byte cp.async for every operand)
    int64_t psi_pad_elems = 0;
    double* d_host_io = nullptr;   // device staging of dmrg_sigma_host (psi, sigma), allocated on first use
    dmrg::TensorMap* d_tmaps = nullptr;   // tensor maps of the TMA path (one per operand matrix and orientation)
    double* d_pack = nullptr;   // packed, N-merged, K-contiguous copies of the R blocks (stage-1 B operands)
    HdItem* d_hd_items = nullptr;
    HdBlock* d_hd_blocks = nullptr;
    int64_t n_hd_blocks = 0;
    HdTile* d_hd_tiles = nullptr;
    int64_t n_hd_tiles = 0;
    double stats[ST_COUNT] = {0};
    // optional per-stage timing
    bool timing = false;
    std::vector<cudaEvent_t> ev;   // 2 per group + 2
    bool timing_valid = false;
    DavidsonWs* dav = nullptr;
    int shard_rank = 0, shard_count = 1;
    const dmrg_comm* comm = nullptr;   // borrowed: all-reduce of the partial sigma / diagonal of a sharded plan
};

namespace dmrg {
void davidson_ws_free(DavidsonWs* ws);
int comm_all_reduce(const dmrg_comm* C, double* buf, int64_t n, cudaStream_t st);
}
