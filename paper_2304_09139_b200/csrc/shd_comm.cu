// shd_comm.cu -- the one exchange step of a particle-sharded evaluation: every rank holds the
// running sums of its own particles' contributions to rho (k_finish1's fold, [tiles][4][1024] double-double pairs);
// they are all-gathered as BYTES in rank order and added on every GPU in that fixed order by k_finish1 itself
// (ncclSum cannot do an error-free double-double add, and a fixed order keeps the result bit-identical on all
// ranks and from run to run).  The minimizers exchange their few double-double dot products the same way.
// NCCL is resolved at run time (dlopen of the libnccl.so.2 that PyTorch has already loaded), so libshd.so has no
// link-time dependency on it and loads on a box without NCCL; a single-GPU handle never touches this file.
#include "../../include/shd.h"
#include "shd_internal.h"

#include <dlfcn.h>
#include <cstring>

namespace {

struct nccl_uid { char internal[128]; };
typedef void* nccl_comm_t;
typedef int (*fn_get_uid)(nccl_uid*);
typedef int (*fn_init_rank)(nccl_comm_t*, int, nccl_uid, int);
typedef int (*fn_allgather)(const void*, void*, size_t, int, nccl_comm_t, cudaStream_t);
typedef int (*fn_destroy)(nccl_comm_t);
typedef const char* (*fn_errstr)(int);

struct nccl_api {
    void* lib = nullptr;
    fn_get_uid get_uid = nullptr;
    fn_init_rank init_rank = nullptr;
    fn_allgather allgather = nullptr;
    fn_destroy destroy = nullptr;
    fn_errstr errstr = nullptr;
};

nccl_api* load_nccl(std::string& err) {
    static nccl_api api;
    if (api.lib) return &api;
    const char* names[] = {"libnccl.so.2", "libnccl.so"};
    for (const char* nm : names) {
        api.lib = dlopen(nm, RTLD_NOW | RTLD_GLOBAL);
        if (api.lib) break;
    }
    if (!api.lib) { err = "NCCL not found (dlopen libnccl.so.2): a sharded handle needs it"; return nullptr; }
    api.get_uid = (fn_get_uid)dlsym(api.lib, "ncclGetUniqueId");
    api.init_rank = (fn_init_rank)dlsym(api.lib, "ncclCommInitRank");
    api.allgather = (fn_allgather)dlsym(api.lib, "ncclAllGather");
    api.destroy = (fn_destroy)dlsym(api.lib, "ncclCommDestroy");
    api.errstr = (fn_errstr)dlsym(api.lib, "ncclGetErrorString");
    if (!api.get_uid || !api.init_rank || !api.allgather || !api.destroy) {
        err = "NCCL symbols missing";
        dlclose(api.lib);
        api.lib = nullptr;
        return nullptr;
    }
    return &api;
}

}  // namespace

struct shd_comm {
    nccl_api* api = nullptr;
    nccl_comm_t comm = nullptr;
};

cudaError_t shd_comm_allgather(shd_ctx* h, const void* send, void* recv, size_t bytes)
{
    if (!h->comm || !h->comm->comm) {
        h->err = "sharded handle without a communicator: call shd_comm_init (or drive the split calls shd_rho_partial / shd_rho_finish / shd_grad_local)";
        return cudaErrorNotReady;
    }
    const int rc = h->comm->api->allgather(send, recv, bytes, /* ncclChar */ 0, h->comm->comm, h->stream);
    if (rc != 0) {
        h->err = std::string("ncclAllGather: ") + (h->comm->api->errstr ? h->comm->api->errstr(rc) : "error");
        return cudaErrorUnknown;
    }
    h->last_launches += 1;
    return cudaSuccess;
}

void shd_comm_free(shd_ctx* h)
{
    if (!h->comm) return;
    if (h->comm->comm) h->comm->api->destroy(h->comm->comm);
    delete h->comm;
    h->comm = nullptr;
}

extern "C" int shd_comm_unique_id(void* id128)
{
    if (!id128) return SHD_EINVAL;
    std::string err;
    nccl_api* api = load_nccl(err);
    if (!api) return SHD_ECUDA;
    nccl_uid id;
    if (api->get_uid(&id) != 0) return SHD_ECUDA;
    std::memcpy(id128, &id, sizeof(id));
    return SHD_OK;
}

extern "C" int shd_comm_init(shd_ctx* h, const void* id128)
{
    if (!h) return SHD_EINVAL;
    if (!id128) { h->err = "NULL pointer"; return SHD_EINVAL; }
    // (a communicator of one rank is allowed: it exercises the same calls on a single GPU)
    if (h->min || h->fire) { h->err = "shd_comm_init: call before the first shd_minimize"; return SHD_EINVAL; }
    nccl_api* api = load_nccl(h->err);
    if (!api) return SHD_ECUDA;
    shd_comm_free(h);
    h->comm = new shd_comm();
    h->comm->api = api;
    nccl_uid id;
    std::memcpy(&id, id128, sizeof(id));
    const int rc = api->init_rank(&h->comm->comm, h->world, id, h->rank);
    if (rc != 0) {
        h->err = std::string("ncclCommInitRank: ") + (api->errstr ? api->errstr(rc) : "error");
        delete h->comm;
        h->comm = nullptr;
        return SHD_ECUDA;
    }
    h->tables_valid = false;             // the gather buffers belong to the sharded setting
    return SHD_OK;
}
