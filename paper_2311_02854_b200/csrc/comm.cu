// dmrg_comm: the one collective of the operator-parallel sigma (the terms mu are partitioned over ranks,
// "NCCL broadcast of the trial vector + reduce of sigma").  Here every rank holds the (replicated, deterministic) Davidson
// vectors, so one H psi needs ONE all-reduce of psi_size doubles: a sharded plan (dmrg_plan_options.shard_*) with a
// communicator attached ends dmrg_sigma / dmrg_hdiag with ncclAllReduce(SUM) enqueued on the caller's stream right behind
// its last launch (the split-K reduce of the last chunk), so the transfer needs no host round trip and dmrg_davidson
// runs unchanged on every rank.  NCCL is loaded at run time (dlopen of the libnccl the process already has -- torch's --
// or the system one): the library has no link-time dependency on it and single-GPU use never touches it.
#include <dlfcn.h>
#include <nccl.h>

#include <new>

#include "plan.h"

struct dmrg_comm {
    ncclComm_t comm = nullptr;
    int rank = 0, world = 1;
};

namespace dmrg {

struct NcclApi {
    void* handle = nullptr;
    ncclResult_t (*GetUniqueId)(ncclUniqueId*) = nullptr;
    ncclResult_t (*CommInitRank)(ncclComm_t*, int, ncclUniqueId, int) = nullptr;
    ncclResult_t (*CommDestroy)(ncclComm_t) = nullptr;
    ncclResult_t (*AllReduce)(const void*, void*, size_t, ncclDataType_t, ncclRedOp_t, ncclComm_t, cudaStream_t) = nullptr;
    const char* (*GetErrorString)(ncclResult_t) = nullptr;
};

static NcclApi* nccl_api() {
    static NcclApi api;
    static bool tried = false;
    if (tried) return api.handle ? &api : nullptr;
    tried = true;
    void* h = dlopen("libnccl.so.2", RTLD_NOW | RTLD_NOLOAD);   // the copy the process already loaded (torch's)
    if (!h) h = dlopen("libnccl.so.2", RTLD_NOW | RTLD_GLOBAL);
    if (!h) h = dlopen("libnccl.so", RTLD_NOW | RTLD_GLOBAL);
    if (!h) { set_error("dmrg_comm: libnccl.so.2 cannot be loaded: %s", dlerror()); return nullptr; }
    api.GetUniqueId = (decltype(api.GetUniqueId))dlsym(h, "ncclGetUniqueId");
    api.CommInitRank = (decltype(api.CommInitRank))dlsym(h, "ncclCommInitRank");
    api.CommDestroy = (decltype(api.CommDestroy))dlsym(h, "ncclCommDestroy");
    api.AllReduce = (decltype(api.AllReduce))dlsym(h, "ncclAllReduce");
    api.GetErrorString = (decltype(api.GetErrorString))dlsym(h, "ncclGetErrorString");
    if (!api.GetUniqueId || !api.CommInitRank || !api.CommDestroy || !api.AllReduce || !api.GetErrorString) {
        set_error("dmrg_comm: libnccl.so.2 lacks an expected symbol");
        dlclose(h);
        return nullptr;
    }
    api.handle = h;
    return &api;
}

// sigma (or the H diagonal) of a sharded plan -> the sum over ranks, in place, on `st`
int comm_all_reduce(const dmrg_comm* C, double* buf, int64_t n, cudaStream_t st) {
    if (!C || !C->comm) return DMRG_OK;
    NcclApi* api = nccl_api();
    if (!api) return DMRG_ECUDA;
    const ncclResult_t r = api->AllReduce(buf, buf, (size_t)n, ncclFloat64, ncclSum, C->comm, st);
    if (r != ncclSuccess) { set_error("dmrg_comm: ncclAllReduce failed: %s", api->GetErrorString(r)); return DMRG_ECUDA; }
    return DMRG_OK;
}

}  // namespace dmrg

using namespace dmrg;

extern "C" {

int dmrg_comm_unique_id(void* id_out, int32_t capacity) {
    if (!id_out || capacity < (int32_t)sizeof(ncclUniqueId)) { set_error("dmrg_comm_unique_id: need a buffer of %d bytes", (int)sizeof(ncclUniqueId)); return DMRG_EINVAL; }
    NcclApi* api = nccl_api();
    if (!api) return DMRG_ECUDA;
    ncclUniqueId id;
    const ncclResult_t r = api->GetUniqueId(&id);
    if (r != ncclSuccess) { set_error("dmrg_comm_unique_id: %s", api->GetErrorString(r)); return DMRG_ECUDA; }
    memcpy(id_out, &id, sizeof id);
    return (int)sizeof id;
}

int dmrg_comm_create(const void* id, int32_t rank, int32_t world, dmrg_comm** out) {
    if (!out) { set_error("dmrg_comm_create: out is NULL"); return DMRG_EINVAL; }
    *out = nullptr;
    if (!id || world < 1 || rank < 0 || rank >= world) { set_error("dmrg_comm_create: bad argument"); return DMRG_EINVAL; }
    NcclApi* api = nccl_api();
    if (!api) return DMRG_ECUDA;
    dmrg_comm* C = new (std::nothrow) dmrg_comm();
    if (!C) { set_error("dmrg_comm_create: out of host memory"); return DMRG_ENOMEM; }
    ncclUniqueId uid;
    memcpy(&uid, id, sizeof uid);
    const ncclResult_t r = api->CommInitRank(&C->comm, world, uid, rank);   // on the calling thread's current device
    if (r != ncclSuccess) { set_error("dmrg_comm_create: ncclCommInitRank failed: %s", api->GetErrorString(r)); delete C; return DMRG_ECUDA; }
    C->rank = rank;
    C->world = world;
    *out = C;
    return DMRG_OK;
}

void dmrg_comm_destroy(dmrg_comm* C) {
    if (!C) return;
    NcclApi* api = nccl_api();
    if (api && C->comm) api->CommDestroy(C->comm);
    delete C;
}

int dmrg_plan_set_comm(dmrg_plan* P, dmrg_comm* C) {
    if (!P) { set_error("dmrg_plan_set_comm: NULL plan"); return DMRG_EINVAL; }
    if (C && (C->world != P->shard_count || C->rank != P->shard_rank)) {
        set_error("dmrg_plan_set_comm: the communicator is rank %d of %d, the plan shard %d of %d", C->rank, C->world, P->shard_rank, P->shard_count);
        return DMRG_EINVAL;
    }
    P->comm = C;
    return DMRG_OK;
}

}  // extern "C"
