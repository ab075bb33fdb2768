// Tensor maps of the TMA path and small planner helpers shared by plan.cu (sigma) and renorm.cu (renormalization).
// Header-only (static functions): not part of the ABI.
#pragma once
#include <cuda.h>   // CUtensorMap types only; the encoder is reached through cudaGetDriverEntryPoint (no libcuda link)

#include <algorithm>
#include <array>
#include <thread>
#include <unordered_map>
#include <vector>

#include "common.h"

namespace dmrg {

// cut a dimension d into full pieces of B plus the remainder.  (Equal-sized pieces were tried and lost: they
// push every tile onto the kernel's ragged path, and the full-tile path is the fast one.)
static inline void cut_dim(int d, int B, std::vector<std::pair<int, int>>& out) {
    out.clear();
    for (int o = 0; o < d; o += B) out.push_back({o, std::min(B, d - o)});
}

// ---- tensor maps of the TMA path -----------------------------------------------------------------------------
// One 2-D FP64 tensor map per operand matrix and orientation.  kind 0: the operand is read k-contiguous (box =
// (GEMM_BK + 4) x tile rows), kind 1: m/n-contiguous (box = (tile + 4) x GEMM_BK): the 4 extra inner columns are the
// bank-conflict padding of the shared-memory tile, written by the TMA unit itself.  Elements outside the matrix
// (inner, outer) are zero-filled by the hardware.
enum MapSpace : uint32_t { MS_OPS = 0, MS_X = 1, MS_PSI = 2, MS_PACK = 3 };
struct MapDesc { uint32_t space; int32_t kind; int64_t off; int32_t inner, outer, ld, box_inner, box_outer; };

// Box of an operand with `k` k-columns per segment and `mn` rows (kind 0) / columns (kind 1) in all:
//   kind 0 (k-contiguous):   inner = min(GEMM_BK, round_up8(k)) + 4 doubles, outer = min(tile, round_up8(mn)) rows
//   kind 1 (m/n-contiguous): inner = min(tile, round_up8(mn)) + 4 doubles,   outer = min(GEMM_BK, round_up4(k)) k-rows
// inner = 4 mod 8 in every case (bank-conflict-free fragment loads); short segments and narrow blocks get small boxes.
struct BoxShape { int inner, outer; };
static inline BoxShape box_shape(int kind, int k, int64_t mn, int tile) {
    const int k8 = std::min(GEMM_BK, (k + 7) & ~7), k4 = std::min(GEMM_BK, (k + 3) & ~3);
    const int mn8 = (int)std::min<int64_t>(tile, (mn + 7) & ~int64_t(7));
    return kind == 0 ? BoxShape{k8 + 4, mn8} : BoxShape{mn8 + 4, k4};
}

struct MapTable {
    std::vector<MapDesc> descs;
    struct KeyHash {
        size_t operator()(const std::array<int64_t, 4>& k) const {
            uint64_t h = 0x9E3779B97F4A7C15ull;
            for (int64_t v : k) h = (h ^ (uint64_t)v) * 0xBF58476D1CE4E5B9ull + (h >> 29);
            return (size_t)h;
        }
    };
    std::unordered_map<std::array<int64_t, 4>, int32_t, KeyHash> index;
    // the X workspace is reused by every chunk, so the same offset can carry matrices of different shapes: the key
    // is the whole descriptor, not the address alone
    int32_t get(uint32_t space, int64_t off, int kind, int inner, int64_t outer, int ld, BoxShape box) {
        const std::array<int64_t, 4> key = {(off << 3) | (int64_t)(space << 1) | kind, ((int64_t)inner << 32) | (uint32_t)ld, outer,
                                            ((int64_t)box.inner << 16) | box.outer};
        auto it = index.find(key);
        if (it != index.end()) return it->second;
        const int32_t id = (int32_t)descs.size();
        descs.push_back({space, kind, off, inner, (int32_t)outer, ld, box.inner, box.outer});
        index.emplace(key, id);
        return id;
    }
};

static inline int encode_tensor_maps(const std::vector<MapDesc>& descs, double* const base[4], std::vector<TensorMap>& out) {
    static_assert(sizeof(TensorMap) == sizeof(CUtensorMap), "TensorMap must be the size of a CUtensorMap");
    typedef CUresult (*EncodeFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                 const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                 CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
    void* fp = nullptr;
    cudaDriverEntryPointQueryResult qres;
    DMRG_CUDA(cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fp, cudaEnableDefault, &qres));
    if (!fp || qres != cudaDriverEntryPointSuccess) { set_error("dmrg_plan_create: cuTensorMapEncodeTiled is not available in this driver"); return DMRG_ECUDA; }
    EncodeFn encode = (EncodeFn)fp;
    out.resize(descs.size());
    // cuTensorMapEncodeTiled is a pure host function: the table (one map per operand matrix, ~1e6 at cfg 5) is
    // encoded by all host threads
    const unsigned nthr = std::max(1u, std::min(32u, std::thread::hardware_concurrency()));
    std::vector<long long> bad(nthr, -1);
    std::vector<int> bad_rc(nthr, 0);
    int dev = 0;
    DMRG_CUDA(cudaGetDevice(&dev));
    auto work = [&](unsigned t) {
        if (t > 0 && cudaSetDevice(dev) != cudaSuccess) { bad[t] = (long long)t; bad_rc[t] = -1; return; }   // the encoder wants a current context
        for (size_t i = t; i < descs.size(); i += nthr) {
            const MapDesc& d = descs[i];
            const cuuint64_t gdim[2] = {(cuuint64_t)d.inner, (cuuint64_t)d.outer};
            const cuuint64_t gstride[1] = {(cuuint64_t)d.ld * 8};
            const cuuint32_t box[2] = {(cuuint32_t)d.box_inner, (cuuint32_t)d.box_outer};
            const cuuint32_t estride[2] = {1, 1};
            const CUresult r = encode((CUtensorMap*)&out[i], CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 2, (void*)(base[d.space] + d.off), gdim, gstride, box,
                                      estride, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
                                      CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
            if (r != CUDA_SUCCESS && bad[t] < 0) { bad[t] = (long long)i; bad_rc[t] = (int)r; }
        }
    };
    std::vector<std::thread> pool;
    for (unsigned t = 1; t < nthr; t++) pool.emplace_back(work, t);
    work(0);
    for (auto& th : pool) th.join();
    for (unsigned t = 0; t < nthr; t++)
        if (bad[t] >= 0) {
            const MapDesc& d = descs[bad[t]];
            set_error("dmrg_plan_create: cuTensorMapEncodeTiled failed (%d) for map %lld: space %u off %lld inner %d outer %d ld %d box %d x %d", bad_rc[t],
                      bad[t], d.space, (long long)d.off, d.inner, d.outer, d.ld, d.box_inner, d.box_outer);
            return DMRG_ECUDA;
        }
    return DMRG_OK;
}


}  // namespace dmrg
