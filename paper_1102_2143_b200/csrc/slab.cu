// slab.cu -- the row (site) partition of SURVEY.md 8(e) / 8(f)-3: every slab owns a contiguous range of rows of A
// and the same range of r, p and every x_k, p_k.  Per iteration the only exchanges are the halo of the vector the
// SpMV gathers (p; for BiCGStab-M also s) and the sums of the fused dot products (2 reals per CG-M iteration,
// 5 complex per BiCGStab-M iteration); the fused multishift update needs no communication at all.
//
//   msolve_slab_plan_*  host only: which columns of a slab's rows live on which other slab, halo numbering, the
//                       slab's matrix with columns renumbered [own rows | halo] -- the part every back end shares
//                       (a rank of a multi-process run builds the plan of its own slab; tests/test_multirank_host.py
//                       checks two ranks' plans against each other over gloo);
//   msolve_slabs_*      P slabs on ONE device, in one process: the halo is written straight into the neighbour's
//                       vector by a gather kernel (the peer-memory store an NVLink domain offers between GPUs; here
//                       the peer is another slab of the same GPU), the dot products are summed over the slabs'
//                       per-CTA partials in fixed slab order.  Every slab runs the SAME kernels as a single handle
//                       (its own msolve_matrix over the renumbered rows), every slab repeats the scalar recurrences
//                       on the same sums, and the whole multi-slab iteration is one WHILE graph.
// Hardware scaling over several GPUs is unmeasured (one GPU per lease); what is shown on one device is that the
// partition, the halo lists and the reductions reproduce the unpartitioned solve.
#include <algorithm>
#include <cstring>
#include <new>
#include <vector>

#include "handle.h"

using namespace msolve;

// ------------------------------------------------------------------------------------------- plan (host)
struct msolve_slab_plan {
    int64_t n = 0;
    int nslabs = 0, rank = 0;
    int64_t row_begin = 0, row_end = 0, nhalo = 0;
    std::vector<int> peer;            // slabs this one receives from, ascending
    std::vector<int64_t> peer_off;    // offset of the peer's entries in the halo (peers ascending, ids ascending)
    std::vector<int32_t> halo_ids;    // GLOBAL column of halo entry j
    std::vector<int32_t> colidx;      // the slab's columns renumbered: own rows 0..nloc-1, halo nloc + j
};

static int owner_of(const int64_t* splits, int nslabs, int64_t c) {
    return (int)(std::upper_bound(splits, splits + nslabs + 1, c) - splits) - 1;
}

extern "C" int msolve_slab_plan_create(msolve_slab_plan** out, int64_t n, int nslabs, const int64_t* h_splits, int rank,
                                       const int32_t* h_rowptr, const int32_t* h_colidx) {
    if (!out) return fail(MSOLVE_EINVAL, "msolve_slab_plan_create: plan is NULL");
    *out = nullptr;
    if (n < 0 || nslabs < 1 || rank < 0 || rank >= nslabs || !h_splits || !h_rowptr) return fail(MSOLVE_EINVAL, "msolve_slab_plan_create: bad argument");
    if (h_splits[0] != 0 || h_splits[nslabs] != n) return fail(MSOLVE_EINVAL, "msolve_slab_plan_create: splits must run from 0 to n");
    for (int p = 0; p < nslabs; ++p)
        if (h_splits[p + 1] < h_splits[p]) return fail(MSOLVE_EINVAL, "msolve_slab_plan_create: splits must not decrease");
    msolve_slab_plan* P = new (std::nothrow) msolve_slab_plan();
    if (!P) return fail(MSOLVE_ENOMEM, "out of host memory");
    P->n = n; P->nslabs = nslabs; P->rank = rank;
    P->row_begin = h_splits[rank]; P->row_end = h_splits[rank + 1];
    const int64_t nloc = P->row_end - P->row_begin;
    if (h_rowptr[0] != 0) { delete P; return fail(MSOLVE_EINVAL, "msolve_slab_plan_create: rowptr must start at 0 (the slab's own rows)"); }
    const int64_t nnz = h_rowptr[nloc];
    if (nnz > 0 && !h_colidx) { delete P; return fail(MSOLVE_EINVAL, "msolve_slab_plan_create: colidx is NULL"); }
    // off-slab columns, unique, ascending: ascending global id is ascending (owner, id), so one sort gives the
    // halo numbering "peers ascending, ids ascending within a peer"
    std::vector<int32_t> off;
    for (int64_t j = 0; j < nnz; ++j) {
        const int64_t c = h_colidx[j];
        if (c < 0 || c >= n) { delete P; return fail(MSOLVE_EINVAL, "msolve_slab_plan_create: column %lld out of range", (long long)c); }
        if (c < P->row_begin || c >= P->row_end) off.push_back((int32_t)c);
    }
    std::sort(off.begin(), off.end());
    off.erase(std::unique(off.begin(), off.end()), off.end());
    P->halo_ids = off;
    P->nhalo = (int64_t)off.size();
    for (int64_t j = 0; j < P->nhalo; ++j) {
        const int o = owner_of(h_splits, nslabs, off[j]);
        if (P->peer.empty() || P->peer.back() != o) { P->peer.push_back(o); P->peer_off.push_back(j); }
    }
    P->peer_off.push_back(P->nhalo);
    P->colidx.resize((size_t)nnz);
    for (int64_t j = 0; j < nnz; ++j) {
        const int64_t c = h_colidx[j];
        if (c >= P->row_begin && c < P->row_end) P->colidx[j] = (int32_t)(c - P->row_begin);
        else P->colidx[j] = (int32_t)(nloc + (std::lower_bound(off.begin(), off.end(), (int32_t)c) - off.begin()));
    }
    *out = P;
    return MSOLVE_OK;
}

extern "C" void msolve_slab_plan_destroy(msolve_slab_plan* P) { delete P; }
extern "C" int64_t msolve_slab_plan_nlocal(const msolve_slab_plan* P) { return P ? P->row_end - P->row_begin : 0; }
extern "C" int64_t msolve_slab_plan_nhalo(const msolve_slab_plan* P) { return P ? P->nhalo : 0; }
extern "C" int msolve_slab_plan_npeers(const msolve_slab_plan* P) { return P ? (int)P->peer.size() : 0; }
extern "C" int msolve_slab_plan_peer(const msolve_slab_plan* P, int j, int* peer_rank, int64_t* halo_offset, int64_t* count,
                                     const int32_t** h_global_ids) {
    if (!P || j < 0 || j >= (int)P->peer.size()) return fail(MSOLVE_EINVAL, "msolve_slab_plan_peer: bad argument");
    if (peer_rank) *peer_rank = P->peer[j];
    if (halo_offset) *halo_offset = P->peer_off[j];
    if (count) *count = P->peer_off[j + 1] - P->peer_off[j];
    if (h_global_ids) *h_global_ids = P->halo_ids.data() + P->peer_off[j];
    return MSOLVE_OK;
}
extern "C" const int32_t* msolve_slab_plan_colidx(const msolve_slab_plan* P) { return P ? P->colidx.data() : nullptr; }

// ------------------------------------------------------------------------------------------- device side
namespace msolve {

// one halo message: `count` elements (times dof) of slab src's vector, rows idx[], go to slab dst's halo at dst_off
struct HaloMsg { int src, dst; int count; int dst_off; const int32_t* idx; };
enum { HALO_P = 0, HALO_S = 1, HALO_SPX = 2 };

// The gather side writes straight into the receiver's vector (peer-memory stores).  grid.y = message.
template <typename E, int DOF>
__global__ void __launch_bounds__(kThreads) k_halo_push(SolveState* const* states, const HaloMsg* msgs, int which) {
    const HaloMsg m = msgs[blockIdx.y];
    const SolveHeader& hs = states[m.src]->h;
    const SolveHeader& hd = states[m.dst]->h;
    if (which != HALO_SPX && states[m.src]->res.done) return;
    const E* src = (const E*)(which == HALO_P ? hs.p : which == HALO_S ? hs.s : hs.sp_x);
    E* dst = (E*)(which == HALO_P ? hd.p : which == HALO_S ? hd.s : const_cast<void*>(hd.sp_x));
    dst += hd.n + (long long)DOF * m.dst_off;
    const int total = m.count * DOF;
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < total; i += gridDim.x * blockDim.x) {
        const int e = i / DOF, c = i - e * DOF;
        dst[i] = src[(long long)DOF * m.idx[e] + c];
    }
}

// Sum of the fused dot products over the slabs: each slab's per-CTA partials in their fixed order, then the slabs
// in slab order; every slab's state receives the total as its only partial (so the unchanged scalar kernels of
// every slab see the global sum).
template <int NACC>
__global__ void __launch_bounds__(kThreads) k_slab_allreduce(SolveState* const* states, int P) {
    __shared__ double red[NACC * 32];
    double total[NACC];
#pragma unroll
    for (int a = 0; a < NACC; ++a) total[a] = 0.0;
    for (int p = 0; p < P; ++p) {
        double s[NACC];
        reduce_partials<NACC>(states[p], s, red);
#pragma unroll
        for (int a = 0; a < NACC; ++a) total[a] += s[a];
    }
    if (threadIdx.x == 0) {
        for (int p = 0; p < P; ++p) {
#pragma unroll
            for (int a = 0; a < NACC; ++a) states[p]->partial[a * kMaxPartials] = total[a];
            states[p]->partial_count = 1;
        }
    }
}

}  // namespace msolve

struct SlabDev {
    msolve_slab_plan* plan = nullptr;
    msolve_matrix* A = nullptr;          // the slab's rows over [own | halo] columns
    int32_t* d_rowptr = nullptr; int32_t* d_colidx = nullptr; void* d_val = nullptr;   // library-owned copies
    int32_t* d_send_idx = nullptr;       // rows of this slab other slabs gather, all messages concatenated
    long long next = 0;                  // vector slot length in elements (own + halo, padded)
};

struct msolve_slabs {
    int P = 0, dtype = MSOLVE_C128, dof = 1;
    int64_t n = 0;                       // scalar rows of the whole matrix
    std::vector<int64_t> splits;         // scalar row ranges
    std::vector<SlabDev> slab;
    SolveState** d_states = nullptr;
    HaloMsg* d_msgs = nullptr;
    int nmsg = 0, max_count = 0;
    cudaStream_t capture_stream = nullptr;
    LoopGraph graphs[2];
    int64_t last_launches = 0;
};

static void slabs_free(msolve_slabs* S) {
    if (!S) return;
    for (int i = 0; i < 2; ++i) {
        if (S->graphs[i].exec) cudaGraphExecDestroy(S->graphs[i].exec);
        if (S->graphs[i].graph) cudaGraphDestroy(S->graphs[i].graph);
    }
    for (SlabDev& d : S->slab) {
        if (d.A) msolve_destroy(d.A);
        if (d.plan) msolve_slab_plan_destroy(d.plan);
        if (d.d_rowptr) cudaFree(d.d_rowptr);
        if (d.d_colidx) cudaFree(d.d_colidx);
        if (d.d_val) cudaFree(d.d_val);
        if (d.d_send_idx) cudaFree(d.d_send_idx);
    }
    if (S->d_states) cudaFree(S->d_states);
    if (S->d_msgs) cudaFree(S->d_msgs);
    if (S->capture_stream) cudaStreamDestroy(S->capture_stream);
    delete S;
}

extern "C" void msolve_slabs_destroy(msolve_slabs* S) { slabs_free(S); }

// rows per slab: multiples of 4 index rows (16-byte aligned slices of b and x for every element type)
static void even_splits(int64_t nrows, int P, std::vector<int64_t>& out) {
    out.resize((size_t)P + 1);
    for (int p = 0; p <= P; ++p) out[p] = std::min<int64_t>(nrows, ((nrows * p / P) + 3) / 4 * 4);
    out[0] = 0; out[P] = nrows;
    for (int p = 1; p <= P; ++p) out[p] = std::max(out[p], out[p - 1]);
}

static int slabs_create(msolve_slabs** out, int dof, int64_t nrows, int64_t nnz, const int32_t* h_rowptr, const int32_t* h_colidx,
                        const void* h_val, int dtype, int nslabs, const int64_t* h_splits, int flags, void* stream) {
    if (!out) return fail(MSOLVE_EINVAL, "msolve_slabs_create: S is NULL");
    *out = nullptr;
    if (nrows < 0 || nnz < 0 || !h_rowptr || (nnz > 0 && (!h_colidx || !h_val))) return fail(MSOLVE_EINVAL, "msolve_slabs_create: bad matrix");
    if (nslabs < 1 || nslabs > 64) return fail(MSOLVE_EINVAL, "msolve_slabs_create: nslabs must be in [1, 64]");
    if (dtype < MSOLVE_C64 || dtype > MSOLVE_F64) return fail(MSOLVE_EINVAL, "msolve_slabs_create: bad dtype");
    if (h_rowptr[0] != 0 || h_rowptr[nrows] != nnz) return fail(MSOLVE_EINVAL, "msolve_slabs_create: rowptr[0] != 0 or rowptr[n] != nnz");
    msolve_slabs* S = new (std::nothrow) msolve_slabs();
    if (!S) return fail(MSOLVE_ENOMEM, "out of host memory");
    S->P = nslabs; S->dtype = dtype; S->dof = dof; S->n = nrows * dof;
    std::vector<int64_t> isplits;                      // in index rows (block rows for BSR3)
    if (h_splits) isplits.assign(h_splits, h_splits + nslabs + 1); else even_splits(nrows, nslabs, isplits);
    const size_t eb = elem_bytes(dtype), vb = (dof == 3 ? 9 : 1) * eb;
    if (isplits[0] != 0 || isplits[nslabs] != nrows) { slabs_free(S); return fail(MSOLVE_EINVAL, "msolve_slabs_create: splits must run from 0 to the number of rows"); }
    for (int p = 0; p < nslabs; ++p)
        if (isplits[p + 1] < isplits[p]) { slabs_free(S); return fail(MSOLVE_EINVAL, "msolve_slabs_create: splits must not decrease"); }
    for (int p = 0; p <= nslabs; ++p) {
        if ((isplits[p] * dof * (int64_t)eb) % 16 != 0 && p < nslabs && p > 0) { slabs_free(S); return fail(MSOLVE_EINVAL, "msolve_slabs_create: split %d is not 16-byte aligned in the vectors", p); }
        S->splits.push_back(isplits[p] * dof);
    }
    S->slab.resize((size_t)nslabs);
    int rc = MSOLVE_OK;
    std::vector<int32_t> rp;
    for (int p = 0; p < nslabs && rc == MSOLVE_OK; ++p) {
        SlabDev& d = S->slab[p];
        const int64_t rb = isplits[p], re = isplits[p + 1], nloc = re - rb;
        rp.resize((size_t)nloc + 1);
        for (int64_t i = 0; i <= nloc; ++i) rp[i] = h_rowptr[rb + i] - h_rowptr[rb];
        const int64_t lnnz = rp[nloc];
        rc = msolve_slab_plan_create(&d.plan, nrows, nslabs, isplits.data(), p, rp.data(), h_colidx + h_rowptr[rb]);
        if (rc != MSOLVE_OK) break;
        if (cudaMalloc((void**)&d.d_rowptr, sizeof(int32_t) * (size_t)(nloc + 1)) != cudaSuccess ||
            cudaMalloc((void**)&d.d_colidx, sizeof(int32_t) * (size_t)std::max<int64_t>(lnnz, 4)) != cudaSuccess ||
            cudaMalloc(&d.d_val, vb * (size_t)std::max<int64_t>(lnnz, 1)) != cudaSuccess) { rc = fail(MSOLVE_ENOMEM, "msolve_slabs_create: cudaMalloc failed"); break; }
        cudaError_t ce = cudaMemcpy(d.d_rowptr, rp.data(), sizeof(int32_t) * (size_t)(nloc + 1), cudaMemcpyHostToDevice);
        if (ce == cudaSuccess && lnnz > 0) ce = cudaMemcpy(d.d_colidx, d.plan->colidx.data(), sizeof(int32_t) * (size_t)lnnz, cudaMemcpyHostToDevice);
        if (ce == cudaSuccess && lnnz > 0) ce = cudaMemcpy(d.d_val, (const char*)h_val + vb * (size_t)h_rowptr[rb], vb * (size_t)lnnz, cudaMemcpyHostToDevice);
        if (ce != cudaSuccess) { rc = fail(MSOLVE_ECUDA, "msolve_slabs_create: copy of slab %d failed: %s", p, cudaGetErrorString(ce)); break; }
        if (dof == 3) rc = msolve_create_bsr3(&d.A, nloc, lnnz, d.d_rowptr, d.d_colidx, d.d_val, dtype, flags, stream);
        else rc = msolve_create_csr(&d.A, nloc, lnnz, d.d_rowptr, d.d_colidx, d.d_val, dtype, flags, stream);
        if (rc != MSOLVE_OK) break;
        d.A->opt.iter_path = 1;                                         // the slab set owns the loop
        d.A->opt.defer = 0;                                             // and runs the step-by-step update (slab_header has no ring)
        d.A->x_stride = S->n;                                           // x_k of a slab is a slice of the global [S][n] array
        d.next = (long long)((((size_t)(nloc + d.plan->nhalo) * dof * eb + 255) / 256 * 256) / eb);
    }
    if (rc != MSOLVE_OK) { slabs_free(S); return rc; }
    // messages: slab q receives plan(q).peer[j] = p's rows halo_ids[...] - row_begin(p)
    std::vector<HaloMsg> msgs;
    std::vector<std::vector<int32_t>> send((size_t)nslabs);
    struct Pending { int src, dst, count, dst_off; size_t idx_off; };
    std::vector<Pending> pend;
    for (int q = 0; q < nslabs; ++q) {
        const msolve_slab_plan* pl = S->slab[q].plan;
        for (size_t j = 0; j < pl->peer.size(); ++j) {
            const int p = pl->peer[j];
            const int64_t o = pl->peer_off[j], c = pl->peer_off[j + 1] - o;
            Pending m{p, q, (int)c, (int)o, send[p].size()};
            for (int64_t t = 0; t < c; ++t) send[p].push_back((int32_t)(pl->halo_ids[o + t] - isplits[p]));
            pend.push_back(m);
            S->max_count = std::max(S->max_count, (int)c);
        }
    }
    for (int p = 0; p < nslabs; ++p) {
        if (send[p].empty()) continue;
        if (cudaMalloc((void**)&S->slab[p].d_send_idx, sizeof(int32_t) * send[p].size()) != cudaSuccess) { slabs_free(S); return fail(MSOLVE_ENOMEM, "msolve_slabs_create: cudaMalloc failed"); }
        cudaMemcpy(S->slab[p].d_send_idx, send[p].data(), sizeof(int32_t) * send[p].size(), cudaMemcpyHostToDevice);
    }
    for (const Pending& m : pend) msgs.push_back(HaloMsg{m.src, m.dst, m.count, m.dst_off, S->slab[m.src].d_send_idx + m.idx_off});
    S->nmsg = (int)msgs.size();
    std::vector<SolveState*> st((size_t)nslabs);
    for (int p = 0; p < nslabs; ++p) st[p] = S->slab[p].A->d_state;
    if (cudaMalloc((void**)&S->d_states, sizeof(SolveState*) * (size_t)nslabs) != cudaSuccess ||
        (S->nmsg && cudaMalloc((void**)&S->d_msgs, sizeof(HaloMsg) * msgs.size()) != cudaSuccess)) { slabs_free(S); return fail(MSOLVE_ENOMEM, "msolve_slabs_create: cudaMalloc failed"); }
    cudaMemcpy(S->d_states, st.data(), sizeof(SolveState*) * (size_t)nslabs, cudaMemcpyHostToDevice);
    if (S->nmsg) cudaMemcpy(S->d_msgs, msgs.data(), sizeof(HaloMsg) * msgs.size(), cudaMemcpyHostToDevice);
    if (cudaStreamCreateWithFlags(&S->capture_stream, cudaStreamNonBlocking) != cudaSuccess || cudaGetLastError() != cudaSuccess) { slabs_free(S); return fail(MSOLVE_ECUDA, "msolve_slabs_create: CUDA error"); }
    *out = S;
    return MSOLVE_OK;
}

extern "C" int msolve_slabs_create_csr(msolve_slabs** out, int64_t n, int64_t nnz, const int32_t* h_rowptr, const int32_t* h_colidx,
                                       const void* h_val, int dtype, int nslabs, const int64_t* h_splits, int flags, void* stream) {
    return slabs_create(out, 1, n, nnz, h_rowptr, h_colidx, h_val, dtype, nslabs, h_splits, flags, stream);
}
extern "C" int msolve_slabs_create_bsr3(msolve_slabs** out, int64_t nbrows, int64_t nblocks, const int32_t* h_browptr, const int32_t* h_bcolidx,
                                        const void* h_blocks, int dtype, int nslabs, const int64_t* h_splits, int flags, void* stream) {
    if (dtype != MSOLVE_C64 && dtype != MSOLVE_C128) return fail(MSOLVE_EINVAL, "msolve_slabs_create_bsr3: dtype must be complex");
    return slabs_create(out, 3, nbrows, nblocks, h_browptr, h_bcolidx, h_blocks, dtype, nslabs, h_splits, flags, stream);
}

extern "C" int msolve_slabs_count(const msolve_slabs* S) { return S ? S->P : 0; }
extern "C" int64_t msolve_slabs_halo_elements(const msolve_slabs* S, int p) { return (S && p >= 0 && p < S->P) ? S->slab[p].plan->nhalo * S->dof : 0; }
extern "C" int64_t msolve_slabs_last_launch_count(const msolve_slabs* S) { return S ? S->last_launches : 0; }

static int base_vectors(int alg) { return alg == MSOLVE_ALG_CGM ? 3 : 5; }

extern "C" size_t msolve_slabs_workspace_bytes(const msolve_slabs* S, int nshifts, int algorithm) {
    if (!S || nshifts < 1 || nshifts > kMaxShifts || (algorithm != MSOLVE_ALG_CGM && algorithm != MSOLVE_ALG_BICGSTABM)) return 0;
    size_t total = 256;
    for (const SlabDev& d : S->slab) total += (size_t)d.next * elem_bytes(S->dtype) * (size_t)(base_vectors(algorithm) + nshifts);
    return total;
}

template <typename E>
static void push_halo_t(const msolve_slabs* S, int which, cudaStream_t s) {
    if (!S->nmsg) return;
    const int gx = std::max(1, std::min(64, (S->max_count * S->dof + kThreads - 1) / kThreads));
    if (S->dof == 3) k_halo_push<E, 3><<<dim3(gx, S->nmsg), kThreads, 0, s>>>(S->d_states, S->d_msgs, which);
    else k_halo_push<E, 1><<<dim3(gx, S->nmsg), kThreads, 0, s>>>(S->d_states, S->d_msgs, which);
}
static void push_halo(const msolve_slabs* S, int which, cudaStream_t s) {
    switch (S->dtype) {
        case MSOLVE_C128: push_halo_t<double2>(S, which, s); break;
        case MSOLVE_C64: push_halo_t<float2>(S, which, s); break;
        case MSOLVE_F64: push_halo_t<double>(S, which, s); break;
        default: push_halo_t<float>(S, which, s); break;
    }
}
static void allreduce(const msolve_slabs* S, int nacc, cudaStream_t s) {
    if (nacc == 1) k_slab_allreduce<1><<<1, kThreads, 0, s>>>(S->d_states, S->P);
    else if (nacc == 2) k_slab_allreduce<2><<<1, kThreads, 0, s>>>(S->d_states, S->P);
    else k_slab_allreduce<5><<<1, kThreads, 0, s>>>(S->d_states, S->P);
}

// kernel launches of one iteration body over all slabs
static int slabs_launches_per_iter(const msolve_slabs* S, int alg) {
    int sp = 0;
    for (const SlabDev& d : S->slab) sp += spmv_launches(d.A);
    const int halo = S->nmsg ? 1 : 0;
    return alg == MSOLVE_ALG_CGM ? 4 * S->P + sp + halo + 2 : 5 * S->P + 2 * sp + 2 * halo + 4;
}

// one iteration body over all slabs (captured into the WHILE graph)
static int slabs_body(const msolve_slabs* S, int alg, cudaStream_t s, cudaGraphConditionalHandle cond, int use_cond, int* count) {
    int rc = MSOLVE_OK, nl = 0;
    auto each_vec = [&](int j, bool with_cond) {
        for (int p = 0; p < S->P && rc == MSOLVE_OK; ++p) { rc = launch_vec_kernel(S->slab[p].A, alg, j, s, cond, with_cond && p == 0 ? use_cond : 0); ++nl; }
    };
    if (alg == MSOLVE_ALG_CGM) {
        each_vec(0, false);                                                    // p <- r + alpha p, own rows
        push_halo(S, HALO_P, s); nl += S->nmsg ? 1 : 0;                        // halo of p
        for (int p = 0; p < S->P && rc == MSOLVE_OK; ++p) { rc = launch_spmv<ROLE_CG>(S->slab[p].A, s); nl += spmv_launches(S->slab[p].A); }
        allreduce(S, 1, s); ++nl;                                              // <p,Ap>
        each_vec(2, false);
        each_vec(3, false);                                                    // fused multishift update: no communication
        allreduce(S, 1, s); ++nl;                                              // |r|^2
        each_vec(4, true);
    } else {
        push_halo(S, HALO_P, s); nl += S->nmsg ? 1 : 0;
        for (int p = 0; p < S->P && rc == MSOLVE_OK; ++p) { rc = launch_spmv<ROLE_B1>(S->slab[p].A, s); nl += spmv_launches(S->slab[p].A); }
        allreduce(S, 2, s); ++nl;                                              // <r0,q>
        each_vec(1, false);
        each_vec(2, false);                                                    // s <- r + beta q
        push_halo(S, HALO_S, s); nl += S->nmsg ? 1 : 0;                        // halo of s
        for (int p = 0; p < S->P && rc == MSOLVE_OK; ++p) { rc = launch_spmv<ROLE_B2>(S->slab[p].A, s); nl += spmv_launches(S->slab[p].A); }
        allreduce(S, 5, s); ++nl;                                              // <t,s>, <t,t>, <r0,t>
        each_vec(4, false);
        each_vec(5, false);
        allreduce(S, 1, s); ++nl;                                              // |r'|^2
        each_vec(6, true);
    }
    if (count) *count = nl;
    return rc;
}

static int slabs_build_graph(msolve_slabs* S, int alg) {
    LoopGraph& g = S->graphs[alg];
    if (g.exec) return MSOLVE_OK;
    MSOLVE_CU(cudaGraphCreate(&g.graph, 0));
    cudaGraphConditionalHandle cond;
    MSOLVE_CU(cudaGraphConditionalHandleCreate(&cond, g.graph, 1, cudaGraphCondAssignDefault));
    cudaGraphNodeParams np = {};
    np.type = cudaGraphNodeTypeConditional;
    np.conditional.handle = cond;
    np.conditional.type = cudaGraphCondTypeWhile;
    np.conditional.size = 1;
    cudaGraphNode_t node;
    MSOLVE_CU(cudaGraphAddNode(&node, g.graph, nullptr, 0, &np));
    cudaGraph_t body = np.conditional.phGraph_out[0];
    MSOLVE_CU(cudaStreamBeginCaptureToGraph(S->capture_stream, body, nullptr, nullptr, 0, cudaStreamCaptureModeThreadLocal));
    const int lrc = slabs_body(S, alg, S->capture_stream, cond, 1, nullptr);
    cudaError_t le = cudaGetLastError();
    cudaGraph_t dummy = nullptr;
    MSOLVE_CU(cudaStreamEndCapture(S->capture_stream, &dummy));
    if (lrc != MSOLVE_OK) return lrc;
    if (le != cudaSuccess) return fail(MSOLVE_ECUDA, "kernel launch during capture failed: %s", cudaGetErrorString(le));
    MSOLVE_CU(cudaGraphInstantiate(&g.exec, g.graph, 0));
    return MSOLVE_OK;
}

// header of slab p for one solve: its rows of b and x (slices of the global arrays), its own vectors in `ws`
static void slab_header(const msolve_slabs* S, int p, int alg, const void* d_b, const double* h_shifts, int nshifts, double tol,
                        int max_iter, void* d_x, char* ws, SolveHeader* h) {
    const SlabDev& d = S->slab[p];
    const size_t eb = elem_bytes(S->dtype);
    const size_t vb = (size_t)d.next * eb;
    memset(h, 0, sizeof(*h));
    h->b = (const char*)d_b + (size_t)S->splits[p] * eb;
    h->x = (char*)d_x + (size_t)S->splits[p] * eb;
    h->r = ws; h->p = ws + vb; h->q = ws + 2 * vb;
    char* next = ws + 3 * vb;
    if (alg == MSOLVE_ALG_BICGSTABM) { h->s = next; h->t = next + vb; next += 2 * vb; }
    h->pk = next;
    h->n = d.A->dev.n;
    h->pk_stride = d.next;
    h->x_stride = S->n;
    h->tol = tol; h->S = nshifts; h->max_iter = max_iter;
    h->stop_rule = d.A->opt.stop_rule;
    for (int k = 0; k < nshifts; ++k) h->sigma[k] = h_shifts[k];
}

static int slabs_solve(int alg, msolve_slabs* S, const void* d_b, const double* h_shifts, int nshifts, double tol, int max_iter,
                       void* d_x, void* d_ws, size_t ws_bytes, int* h_iterations, int* h_conv_iter, double* h_relres, void* stream_) {
    if (!S) return fail(MSOLVE_EINVAL, "msolve_slabs solve: S is NULL");
    if (nshifts < 1 || nshifts > kMaxShifts) return fail(MSOLVE_EINVAL, "msolve_slabs solve: nshifts must be in [1, %d]", kMaxShifts);
    if (!d_b || !d_x || !h_shifts || !d_ws) return fail(MSOLVE_EINVAL, "msolve_slabs solve: NULL argument");
    if (!(tol >= 0.0) || max_iter < 0) return fail(MSOLVE_EINVAL, "msolve_slabs solve: bad tol / max_iter");
    if (((uintptr_t)d_b & 15u) || ((uintptr_t)d_x & 15u)) return fail(MSOLVE_EINVAL, "msolve_slabs solve: d_b / d_x must be 16-byte aligned");
    const size_t need = msolve_slabs_workspace_bytes(S, nshifts, alg);
    if (ws_bytes < need) return fail(MSOLVE_ENOMEM, "msolve_slabs solve: workspace too small (%zu < %zu)", ws_bytes, need);
    int rc = check_device(S->slab[0].A, "msolve_slabs solve");
    if (rc != MSOLVE_OK) return rc;
    cudaStream_t stream = (cudaStream_t)stream_;
    const size_t eb = elem_bytes(S->dtype);
    const size_t xbytes = (size_t)nshifts * (size_t)S->n * eb;
    if (S->n == 0 || max_iter == 0) {
        MSOLVE_CU(cudaMemsetAsync(d_x, 0, xbytes, stream));
        MSOLVE_CU(cudaStreamSynchronize(stream));
        if (h_iterations) *h_iterations = 0;
        for (int k = 0; k < nshifts; ++k) { if (h_conv_iter) h_conv_iter[k] = S->n == 0 ? 0 : -1; if (h_relres) h_relres[k] = S->n == 0 ? 0.0 : 1.0; }
        S->last_launches = 0;
        return S->n == 0 ? MSOLVE_OK : MSOLVE_MAXITER;
    }
    rc = slabs_build_graph(S, alg);
    if (rc != MSOLVE_OK) return rc;
    char* ws = (char*)(((uintptr_t)d_ws + 255) / 256 * 256);
    for (int p = 0; p < S->P; ++p) {
        msolve_matrix* A = S->slab[p].A;
        slab_header(S, p, alg, d_b, h_shifts, nshifts, tol, max_iter, d_x, ws, &A->h_stage->h);
        SolveResult* r = &A->h_stage->res;
        memset(r, 0, sizeof(*r));
        r->nactive = nshifts;
        for (int k = 0; k < kMaxShifts; ++k) { r->conv_iter[k] = -1; r->relres[k] = 1.0; }
        MSOLVE_CU(cudaMemcpyAsync(A->d_state, A->h_stage, sizeof(SolveHeader) + sizeof(SolveResult), cudaMemcpyHostToDevice, stream));
        ws += (size_t)S->slab[p].next * eb * (size_t)(base_vectors(alg) + nshifts);
    }
    // init: r <- b, p <- b on every slab, <b,b> summed over the slabs, scalars
    for (int p = 0; p < S->P; ++p) if ((rc = launch_init_vectors(S->slab[p].A, stream)) != MSOLVE_OK) return rc;
    allreduce(S, 1, stream);
    for (int p = 0; p < S->P; ++p) if ((rc = launch_init_state(S->slab[p].A, stream)) != MSOLVE_OK) return rc;
    MSOLVE_CU(cudaGetLastError());
    MSOLVE_CU(cudaGraphLaunch(S->graphs[alg].exec, stream));
    SolveResult* hr = &S->slab[0].A->h_stage->res;      // every slab ends with the same result block
    MSOLVE_CU(cudaMemcpyAsync(hr, &S->slab[0].A->d_state->res, sizeof(SolveResult), cudaMemcpyDeviceToHost, stream));
    MSOLVE_CU(cudaStreamSynchronize(stream));
    if (hr->zero_rhs || (hr->status == MSOLVE_BREAKDOWN && hr->n_iter == 0)) {
        MSOLVE_CU(cudaMemsetAsync(d_x, 0, xbytes, stream));
        MSOLVE_CU(cudaStreamSynchronize(stream));
    }
    S->last_launches = 2 * S->P + 1 + (int64_t)slabs_launches_per_iter(S, alg) * std::max(1, hr->n_iter + (hr->status == MSOLVE_BREAKDOWN ? 1 : 0));
    if (h_iterations) *h_iterations = hr->n_iter;
    for (int k = 0; k < nshifts; ++k) {
        if (h_conv_iter) h_conv_iter[k] = hr->conv_iter[k];
        if (h_relres) h_relres[k] = hr->relres[k];
    }
    return hr->status;
}

extern "C" int msolve_slabs_cgm(msolve_slabs* S, const void* d_b, const double* h_shifts, int nshifts, double tol, int max_iter,
                                void* d_x, void* d_workspace, size_t workspace_bytes, int* h_iterations, int* h_conv_iter,
                                double* h_relres, void* stream) {
    return slabs_solve(MSOLVE_ALG_CGM, S, d_b, h_shifts, nshifts, tol, max_iter, d_x, d_workspace, workspace_bytes, h_iterations, h_conv_iter, h_relres, stream);
}
extern "C" int msolve_slabs_bicgstabm(msolve_slabs* S, const void* d_b, const double* h_shifts, int nshifts, double tol, int max_iter,
                                      void* d_x, void* d_workspace, size_t workspace_bytes, int* h_iterations, int* h_conv_iter,
                                      double* h_relres, void* stream) {
    return slabs_solve(MSOLVE_ALG_BICGSTABM, S, d_b, h_shifts, nshifts, tol, max_iter, d_x, d_workspace, workspace_bytes, h_iterations, h_conv_iter, h_relres, stream);
}

// y = A x over the slabs with the halo exchange (tests): x and y are global vectors of n elements; `d_workspace`
// holds the slabs' [own | halo] copies of x (msolve_slabs_workspace_bytes(S, 1, CGM) is enough).
extern "C" int msolve_slabs_spmv(msolve_slabs* S, const void* d_x, void* d_y, void* d_workspace, size_t workspace_bytes, double* h_dot, void* stream_) {
    if (!S || !d_x || !d_y || !d_workspace) return fail(MSOLVE_EINVAL, "msolve_slabs_spmv: NULL argument");
    if (workspace_bytes < msolve_slabs_workspace_bytes(S, 1, MSOLVE_ALG_CGM)) return fail(MSOLVE_ENOMEM, "msolve_slabs_spmv: workspace too small");
    cudaStream_t stream = (cudaStream_t)stream_;
    const size_t eb = elem_bytes(S->dtype);
    char* ws = (char*)(((uintptr_t)d_workspace + 255) / 256 * 256);
    int rc;
    for (int p = 0; p < S->P; ++p) {
        msolve_matrix* A = S->slab[p].A;
        SolveHeader* h = &A->h_stage->h;
        memset(h, 0, sizeof(*h));
        const size_t nloc_b = (size_t)A->dev.n * eb;
        MSOLVE_CU(cudaMemcpyAsync(ws, (const char*)d_x + (size_t)S->splits[p] * eb, nloc_b, cudaMemcpyDeviceToDevice, stream));
        h->sp_x = ws; h->sp_u = ws; h->sp_y = (char*)d_y + (size_t)S->splits[p] * eb; h->n = A->dev.n; h->S = 1;
        memset(&A->h_stage->res, 0, sizeof(SolveResult));
        MSOLVE_CU(cudaMemcpyAsync(A->d_state, A->h_stage, sizeof(SolveHeader) + sizeof(SolveResult), cudaMemcpyHostToDevice, stream));
        ws += (size_t)S->slab[p].next * eb * 4;
    }
    push_halo(S, HALO_SPX, stream);
    for (int p = 0; p < S->P; ++p) if (S->slab[p].A->dev.n > 0 && (rc = launch_spmv<ROLE_GEN>(S->slab[p].A, stream)) != MSOLVE_OK) return rc;
    allreduce(S, 2, stream);
    MSOLVE_CU(cudaGetLastError());
    double tmp[2] = {0.0, 0.0};
    MSOLVE_CU(cudaMemcpyAsync(&tmp[0], &S->slab[0].A->d_state->partial[0], sizeof(double), cudaMemcpyDeviceToHost, stream));
    MSOLVE_CU(cudaMemcpyAsync(&tmp[1], &S->slab[0].A->d_state->partial[kMaxPartials], sizeof(double), cudaMemcpyDeviceToHost, stream));
    MSOLVE_CU(cudaStreamSynchronize(stream));
    if (h_dot) { h_dot[0] = tmp[0]; h_dot[1] = tmp[1]; }
    return MSOLVE_OK;
}
