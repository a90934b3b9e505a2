// Row e: the exchange step of the row-sharded solve (Fig. 2; Algorithm 3
// lines 8, 12, 16).  Every rank holds a star-aligned block of rows as an ordinary local
// matrix; the attitude + instrumental + global slice of the n-vectors is replicated and summed
// over the ranks with ncclAllReduce (the paper does it with MPI_Reduce through host memory).
// NCCL is loaded with dlopen at gsr_comm_create, so that the library has no link-time
// dependency on it and single-GPU users never touch it.
#include <dlfcn.h>
#include <nccl.h>
#include <string.h>

#include <new>

#include "gsr_internal.h"

struct gsr_comm {
    void* lib;
    ncclComm_t comm;
    int rank, world;
    ncclResult_t (*AllReduce)(const void*, void*, size_t, ncclDataType_t, ncclRedOp_t, ncclComm_t,
                              cudaStream_t);
    ncclResult_t (*CommDestroy)(ncclComm_t);
};

namespace gsr {

static void* open_nccl() {
    // torch has normally loaded its own libnccl.so.2 already: the soname resolves to that copy
    void* h = dlopen("libnccl.so.2", RTLD_NOW | RTLD_GLOBAL);
    if (!h) h = dlopen("libnccl.so", RTLD_NOW | RTLD_GLOBAL);
    return h;
}

int comm_allreduce_sum(gsr_comm* c, double* buf, size_t count, cudaStream_t s) {
    if (!c || count == 0) return GSR_OK;
    if (c->AllReduce(buf, buf, count, ncclDouble, ncclSum, c->comm, s) != ncclSuccess) return GSR_ECUDA;
    return GSR_OK;
}

}  // namespace gsr

extern "C" {

int gsr_comm_unique_id(void* id_out, int64_t bytes) {
    if (!id_out || bytes < (int64_t)sizeof(ncclUniqueId)) return GSR_EINVAL;
    void* h = gsr::open_nccl();
    if (!h) return GSR_EUNSUPPORTED;
    auto fn = (ncclResult_t(*)(ncclUniqueId*))dlsym(h, "ncclGetUniqueId");
    if (!fn) return GSR_EUNSUPPORTED;
    ncclUniqueId id;
    if (fn(&id) != ncclSuccess) return GSR_ECUDA;
    memcpy(id_out, &id, sizeof(id));
    return GSR_OK;
}

int gsr_comm_create(gsr_comm** out, int rank, int world, const void* id_in, int64_t bytes) {
    if (!out) return GSR_EINVAL;
    *out = nullptr;
    if (!id_in || bytes < (int64_t)sizeof(ncclUniqueId) || world < 1 || rank < 0 || rank >= world)
        return GSR_EINVAL;
    void* h = gsr::open_nccl();
    if (!h) return GSR_EUNSUPPORTED;
    auto init = (ncclResult_t(*)(ncclComm_t*, int, ncclUniqueId, int))dlsym(h, "ncclCommInitRank");
    gsr_comm* c = new (std::nothrow) gsr_comm();
    if (!c) return GSR_ENOMEM;
    c->lib = h;
    c->rank = rank;
    c->world = world;
    c->AllReduce = (decltype(c->AllReduce))dlsym(h, "ncclAllReduce");
    c->CommDestroy = (decltype(c->CommDestroy))dlsym(h, "ncclCommDestroy");
    if (!init || !c->AllReduce || !c->CommDestroy) {
        delete c;
        return GSR_EUNSUPPORTED;
    }
    ncclUniqueId id;
    memcpy(&id, id_in, sizeof(id));
    if (init(&c->comm, world, id, rank) != ncclSuccess) {
        delete c;
        return GSR_ECUDA;
    }
    *out = c;
    return GSR_OK;
}

int gsr_comm_destroy(gsr_comm* c) {
    if (!c) return GSR_OK;
    c->CommDestroy(c->comm);
    delete c;
    return GSR_OK;
}

int gsr_matrix_set_comm(gsr_matrix* A, gsr_comm* c, int64_t n_rows_global, int64_t n_cols_global) {
    if (!A) return GSR_EINVAL;
    if (A->state != 1 || A->p != nullptr || A->ws.st != nullptr) return GSR_ESTATE;   // before precondition / solve
    // constraint rows (row f3) stay with the rank whose handle they were given to, in LOCAL
    // column numbering; n_rows_global counts them too (every rank's)
    if (c && (n_rows_global < A->dims.n_rows + A->n_con || n_cols_global < A->n_cols)) return GSR_EINVAL;
    A->comm = c;
    A->m_global = c ? n_rows_global : A->dims.n_rows + A->n_con;
    A->n_global = c ? n_cols_global : A->n_cols;
    return GSR_OK;
}

}  // extern "C"
