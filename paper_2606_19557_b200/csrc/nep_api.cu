// nep_api.cu -- C ABI entry points of libnep_b200 (include/nep.h): argument checks, state machine,
// host<->device marshalling.  All arithmetic of the step lives in the kernels of the other .cu files.
#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <algorithm>
#include <new>

#include "nep_kernels.cuh"

static thread_local std::string g_create_error;

namespace nep {

int fail(nep_ctx* c, int code, const std::string& msg)
{
    if (c) c->err = msg; else g_create_error = msg;
    return code;
}

void* dev_alloc(nep_ctx* c, size_t bytes)
{
    if (bytes == 0) bytes = 256;
    void* p = c->alloc(c->user, bytes);   // the library never calls cudaMalloc: device memory is the caller's (include/nep.h)
    if (!p) { c->err = "device allocation of " + std::to_string(bytes) + " bytes failed"; return nullptr; }
    c->allocs.push_back(p);
    return p;
}

void dev_free(nep_ctx* c, void* p)
{
    if (!p) return;
    auto it = std::find(c->allocs.begin(), c->allocs.end(), p);
    if (it != c->allocs.end()) c->allocs.erase(it);
    c->free_(c->user, p);
}

void prof_begin(nep_ctx* c, const char* name)
{
    ++c->launches;
    if (!c->prof.on || c->prof.paused) return;
    Profiler::Rec r; r.name = name;
    auto get = [&]() { cudaEvent_t e; if (!c->prof.pool.empty()) { e = c->prof.pool.back(); c->prof.pool.pop_back(); } else cudaEventCreate(&e); return e; };
    r.a = get(); r.b = get();
    cudaEventRecord(r.a, c->stream);
    c->prof.pending.push_back(r);
}
void prof_end(nep_ctx* c)
{
    if (!c->prof.on || c->prof.paused) return;
    cudaEventRecord(c->prof.pending.back().b, c->stream);
}

}  // namespace nep

using namespace nep;

#define CHECK_CTX(c) do { if (!(c)) return NEP_EINVAL; } while (0)
#define ALLOC(c, ptr, type, count)                                              \
    do {                                                                        \
        (ptr) = (type*)dev_alloc((c), sizeof(type) * (size_t)(count));          \
        if (!(ptr)) return NEP_ENOMEM;                                          \
    } while (0)

template <class T>
static int upload(nep_ctx* c, T*& dptr, const T* h, size_t count)
{
    dptr = (T*)dev_alloc(c, sizeof(T) * std::max<size_t>(count, 1));
    if (!dptr) return NEP_ENOMEM;
    if (count) NEP_CUDA(c, cudaMemcpyAsync(dptr, h, sizeof(T) * count, cudaMemcpyHostToDevice, c->stream));
    return NEP_OK;
}

namespace nep {
// Per-slot tables of the current slot order (h_slot_of): species and rank among the same species per slot, the atom of
// every slot and the slot of every atom; the force labels follow if they are loaded.
int upload_slot_tables(nep_ctx* c)
{
    c->batch_tables_valid = false;     // the type-sorted atom list of a batch depends on the slot order
    ++c->graph_gen;                    // the tables move to new buffers: a captured step graph points at the old ones
    DataDev& d = c->d;
    const int T = c->m.T;
    std::vector<int> type_p((size_t)c->NP, -1), rank_p((size_t)c->NP, 0), orig_p((size_t)c->NP, -1);
    for (int s = 0; s < c->S; ++s) {
        const int64_t a0 = c->h_aoff[s], p0 = c->h_pbase[s];
        for (int i = 0; i < c->h_nat[s]; ++i) { const int sl = c->h_slot_of[a0 + i]; orig_p[p0 + sl] = i; type_p[p0 + sl] = c->h_type[a0 + i]; }
        std::vector<int> tc(T, 0);
        for (int sl = 0; sl < c->h_nat[s]; ++sl) rank_p[p0 + sl] = tc[type_p[p0 + sl]]++;
    }
    const void* olds[] = { d.type_p, d.rank_p, d.orig_p, d.slot_of };
    for (const void* p : olds) dev_free(c, const_cast<void*>(p));
    d.type_p = d.rank_p = d.orig_p = d.slot_of = nullptr;
    int *dtp, *drk, *dor, *dso;
    int rc;
    if ((rc = upload<int>(c, dtp, type_p.data(), type_p.size()))) return rc;
    if ((rc = upload<int>(c, drk, rank_p.data(), rank_p.size()))) return rc;
    if ((rc = upload<int>(c, dor, orig_p.data(), orig_p.size()))) return rc;
    if ((rc = upload<int>(c, dso, c->h_slot_of.data(), c->h_slot_of.size()))) return rc;
    d.type_p = dtp; d.rank_p = drk; d.orig_p = dor; d.slot_of = dso;
    if (c->have_labels && !c->h_Flab.empty()) {
        std::vector<float> Fp((size_t)3 * c->NP, 0.0f);
        for (int s = 0; s < c->S; ++s)
            for (int i = 0; i < c->h_nat[s]; ++i)
                for (int k = 0; k < 3; ++k) {
                    const int64_t p = c->h_pbase[s] + c->h_slot_of[c->h_aoff[s] + i];
                    Fp[(size_t)((p / WARP) * 3 + k) * WARP + p % WARP] = c->h_Flab[3 * (c->h_aoff[s] + i) + k];
                }
        NEP_CUDA(c, cudaMemcpyAsync(const_cast<float*>(d.Flab), Fp.data(), 4 * Fp.size(), cudaMemcpyHostToDevice, c->stream));
    }
    NEP_CUDA(c, cudaStreamSynchronize(c->stream));
    return NEP_OK;
}
}  // namespace nep

extern "C" {

const char* nep_version(void) { return "nep_b200 0.2 (sm_100a, fp32 step, fp64 neighbour predicate)"; }

const char* nep_last_error(const nep_ctx* ctx) { return ctx ? ctx->err.c_str() : g_create_error.c_str(); }

int nep_create(nep_ctx** out, int n_species, double rc_R, double rc_A, int n_max_R, int n_max_A, int basis_R, int basis_A,
               int l_max_3b, int l_max_4b, int l_max_5b, int neurons, nep_alloc_fn alloc, nep_free_fn free_, void* alloc_user,
               void* cuda_stream)
{
    if (!out) return fail(nullptr, NEP_EINVAL, "out is NULL");
    *out = nullptr;
    if (n_species < 1 || n_species > MAX_T) return fail(nullptr, NEP_EINVAL, "n_species must be in 1..16");
    if (!(rc_A > 0.0) || !(rc_A <= rc_R) || !std::isfinite(rc_R)) return fail(nullptr, NEP_EINVAL, "need 0 < rc_A <= rc_R");
    if (n_max_R < 0 || n_max_A < 0 || n_max_R > 19 || n_max_A > 19) return fail(nullptr, NEP_EINVAL, "n_max must be in 0..19");
    if (basis_R < 1 || basis_A < 1 || basis_R > 16 || basis_A > 16) return fail(nullptr, NEP_EINVAL, "basis_size must be in 1..16");
    if (l_max_3b < 1 || l_max_3b > 4) return fail(nullptr, NEP_EINVAL, "l_max_3b must be in 1..4");
    if (!(l_max_4b == 0 || l_max_4b == 2)) return fail(nullptr, NEP_EINVAL, "l_max_4b must be 0 or 2");
    if (!(l_max_5b == 0 || l_max_5b == 1)) return fail(nullptr, NEP_EINVAL, "l_max_5b must be 0 or 1");
    if (neurons < 1 || neurons > 512) return fail(nullptr, NEP_EINVAL, "neurons must be in 1..512");
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) {
        cudaGetLastError();
        return fail(nullptr, NEP_ECUDA, "no CUDA device: libnep_b200 has no CPU fallback");
    }
    if (alloc == nullptr || free_ == nullptr) return fail(nullptr, NEP_EINVAL, "alloc and free_ are required: the library does not allocate device memory itself");
    nep_ctx* c = new (std::nothrow) nep_ctx();
    if (!c) return fail(nullptr, NEP_ENOMEM, "host allocation failed");
    c->rcR = rc_R; c->rcA = rc_A; c->n_max_R = n_max_R; c->n_max_A = n_max_A; c->basis_R = basis_R; c->basis_A = basis_A;
    c->l3 = l_max_3b; c->l4 = l_max_4b; c->l5 = l_max_5b;
    c->alloc = alloc; c->free_ = free_; c->user = alloc_user; c->stream = (cudaStream_t)cuda_stream;
    ModelDev& m = c->m;
    m.T = n_species; m.nR = n_max_R + 1; m.nA = n_max_A + 1; m.KR = basis_R + 1; m.KA = basis_A + 1; m.KRP = (m.KR + 3) & ~3;
    m.H = neurons; m.has4 = l_max_4b > 0; m.has5 = l_max_5b > 0; m.l3 = l_max_3b; m.nang = m.l3 + m.has4 + m.has5;
    m.D = m.nR + m.nA * m.nang; m.DP = (m.D + 7) & ~7; m.HP = (m.H + 7) & ~7;
    m.rcR = (float)rc_R; m.rcA = (float)rc_A; m.rcinvR = (float)(1.0 / rc_R); m.rcinvA = (float)(1.0 / rc_A);
    m.per_type = (m.D + 2) * m.H; m.o_b1 = m.per_type * m.T; m.o_cR = m.o_b1 + 1; m.o_cA = m.o_cR + m.T * m.T * m.nR * m.KR;
    m.npar = m.o_cA + m.T * m.T * m.nA * m.KA;
    int dev = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&c->sm_count, cudaDevAttrMultiProcessorCount, dev);
    cudaDeviceGetAttribute(&c->max_smem_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
    cudaDeviceGetAttribute(&c->max_smem_sm, cudaDevAttrMaxSharedMemoryPerMultiprocessor, dev);
    if (cudaMallocHost(&c->h_small, sizeof c->h_small_bytes) != cudaSuccess) { c->h_small = nullptr; cudaGetLastError(); }
    {   // network kernels: tensor-core tiles when they fit; NEP_ANN_FFMA=1 selects the FFMA tiles (measurement aid)
        const char* e = getenv("NEP_ANN_FFMA");
        c->ann_tc = !(e && e[0] == '1') && ann_tc_fits(c, false) && ann_tc_fits(c, true);
    }
    size_t np = (size_t)m.npar;
    c->theta = (float*)dev_alloc(c, 4 * np); c->g = (float*)dev_alloc(c, 4 * np); c->am = (float*)dev_alloc(c, 4 * np);
    c->av = (float*)dev_alloc(c, 4 * np); c->avmax = (float*)dev_alloc(c, 4 * np); c->scaler = (float*)dev_alloc(c, 4 * (size_t)m.DP);
    if (!c->theta || !c->g || !c->am || !c->av || !c->avmax || !c->scaler) {
        g_create_error = c->err; nep_destroy(c); return NEP_ENOMEM;
    }
    cudaMemsetAsync(c->g, 0, 4 * np, c->stream); cudaMemsetAsync(c->am, 0, 4 * np, c->stream);
    cudaMemsetAsync(c->av, 0, 4 * np, c->stream); cudaMemsetAsync(c->avmax, 0, 4 * np, c->stream);
    cudaMemsetAsync(c->theta, 0, 4 * np, c->stream);
    if (cudaStreamSynchronize(c->stream) != cudaSuccess) {
        g_create_error = std::string("CUDA error in nep_create: ") + cudaGetErrorString(cudaGetLastError());
        nep_destroy(c); return NEP_ECUDA;
    }
    *out = c;
    return NEP_OK;
}

int nep_destroy(nep_ctx* c)
{
    if (!c) return NEP_OK;
    cudaStreamSynchronize(c->stream);
    graph_drop(c);
    if (c->cap_stream) cudaStreamDestroy(c->cap_stream);
    if (c->side_stream) cudaStreamDestroy(c->side_stream);
    if (c->ev_fork) cudaEventDestroy(c->ev_fork);
    if (c->ev_join) cudaEventDestroy(c->ev_join);
    std::vector<void*> a = c->allocs;
    for (void* p : a) dev_free(c, p);
    if (c->h_stage) cudaFreeHost(c->h_stage);
    if (c->h_small) cudaFreeHost(c->h_small);
    for (auto& r : c->prof.pending) { cudaEventDestroy(r.a); cudaEventDestroy(r.b); }
    for (auto e : c->prof.pool) cudaEventDestroy(e);
    delete c;
    return NEP_OK;
}

int nep_num_descriptors(const nep_ctx* c) { return c ? c->m.D : NEP_EINVAL; }
int64_t nep_num_params(const nep_ctx* c) { return c ? c->m.npar : NEP_EINVAL; }

static void free_dataset(nep_ctx* c)
{
    DataDev& d = c->d;
    const void* ptrs[] = { d.pos, d.box, d.type, d.atom_off, d.pbase, d.type_p, d.rank_p, d.orig_p, d.slot_of, d.slice_struct, d.Elab, d.Flab, d.Wlab, d.hasv,
                           d.offR, d.jR, d.shR, d.offA, d.jA, d.shA, d.cntR, d.recoffR, d.recR, d.cntA, d.recoffA, d.recA, d.B };
    for (const void* p : ptrs) dev_free(c, const_cast<void*>(p));
    memset(&d, 0, sizeof d);
    c->have_data = c->have_labels = c->have_nbrs = c->forward_valid = c->grad_valid = c->loss_valid = false;
    c->batch_tables_valid = false;
    ++c->graph_gen;
}

static int upload_labels(nep_ctx* c, const double* E, const double* F, const double* W, const unsigned char* hv)
{
    DataDev& d = c->d;
    // validate before anything is released: a rejected call leaves the previous labels in place
    for (int64_t i = 0; i < c->S; ++i) if (!std::isfinite(E[i])) return fail(c, NEP_EINVAL, "non-finite energy label");
    for (int64_t i = 0; i < 3 * c->N; ++i) if (!std::isfinite(F[i])) return fail(c, NEP_EINVAL, "non-finite force label");
    for (int64_t i = 0; i < 9 * (int64_t)c->S; ++i) if (!std::isfinite(W[i])) return fail(c, NEP_EINVAL, "non-finite virial label");
    std::vector<float> hF((size_t)3 * c->N), Fp((size_t)3 * c->NP, 0.0f), Wf((size_t)9 * c->S);
    for (int64_t i = 0; i < 3 * c->N; ++i) hF[i] = (float)F[i];
    for (int s = 0; s < c->S; ++s)
        for (int i = 0; i < c->h_nat[s]; ++i)
            for (int k = 0; k < 3; ++k) {   // slice-blocked [slice][3][32], slot order
                const int64_t p = c->h_pbase[s] + c->h_slot_of[c->h_aoff[s] + i];
                Fp[(size_t)((p / WARP) * 3 + k) * WARP + p % WARP] = hF[3 * (c->h_aoff[s] + i) + k];
            }
    for (size_t i = 0; i < Wf.size(); ++i) Wf[i] = (float)W[i];
    std::vector<unsigned char> hasv((size_t)c->S, 1);
    if (hv) for (int s = 0; s < c->S; ++s) hasv[s] = hv[s] ? 1 : 0;
    // upload into new buffers; the old ones are swapped out and released only after every copy has succeeded
    double* dE = nullptr; float *dF = nullptr, *dW = nullptr; unsigned char* dh = nullptr;
    int rc;
    if ((rc = upload<double>(c, dE, E, c->S)) || (rc = upload<float>(c, dF, Fp.data(), Fp.size())) ||
        (rc = upload<float>(c, dW, Wf.data(), Wf.size())) || (rc = upload<unsigned char>(c, dh, hasv.data(), c->S)) ||
        (cudaStreamSynchronize(c->stream) != cudaSuccess && (rc = fail(c, NEP_ECUDA, "label upload failed")))) {
        dev_free(c, dE); dev_free(c, dF); dev_free(c, dW); dev_free(c, dh);
        return rc;
    }
    dev_free(c, (void*)d.Elab); dev_free(c, (void*)d.Flab); dev_free(c, (void*)d.Wlab); dev_free(c, (void*)d.hasv);
    d.Elab = dE; d.Flab = dF; d.Wlab = dW; d.hasv = dh;
    c->h_Flab.swap(hF); c->h_hasv.swap(hasv);
    ++c->graph_gen;
    c->have_labels = true;
    c->grad_valid = false;
    return NEP_OK;
}

int nep_load_structures(nep_ctx* c, int S, const int* n_atoms, const double* pos, const double* box, const int* type,
                        const double* E, const double* F, const double* W, const unsigned char* has_virial)
{
    CHECK_CTX(c);
    if (S < 0 || (S > 0 && (!n_atoms || !pos || !box || !type))) return fail(c, NEP_EINVAL, "NULL input array");
    bool lab = E || F || W;
    if (lab && !(E && F && W)) return fail(c, NEP_EINVAL, "E, F and W must be given together");
    std::vector<int64_t> aoff(S + 1, 0), pbase(S + 1, 0);
    for (int s = 0; s < S; ++s) {
        if (n_atoms[s] < 1) return fail(c, NEP_EINVAL, "structure with no atoms");
        aoff[s + 1] = aoff[s] + n_atoms[s];
        pbase[s + 1] = pbase[s] + ((n_atoms[s] + WARP - 1) / WARP) * WARP;
    }
    int64_t N = aoff[S], NP = pbase[S];
    if (NP / WARP > (int64_t)INT32_MAX / 4) return fail(c, NEP_ECAPACITY, "too many atoms");
    for (int s = 0; s < S; ++s) {
        const double* b = box + 9 * s;
        for (int k = 0; k < 9; ++k) if (!std::isfinite(b[k])) return fail(c, NEP_EINVAL, "non-finite box");
        double det = b[0] * (b[4] * b[8] - b[5] * b[7]) - b[1] * (b[3] * b[8] - b[5] * b[6]) + b[2] * (b[3] * b[7] - b[4] * b[6]);
        if (!(det > 0.0)) return fail(c, NEP_EINVAL, "det(box) <= 0 for structure " + std::to_string(s));
        // inverse (columns = reciprocal vectors / det): frac = r . inv
        double inv[9] = { (b[4] * b[8] - b[5] * b[7]) / det, (b[2] * b[7] - b[1] * b[8]) / det, (b[1] * b[5] - b[2] * b[4]) / det,
                          (b[5] * b[6] - b[3] * b[8]) / det, (b[0] * b[8] - b[2] * b[6]) / det, (b[2] * b[3] - b[0] * b[5]) / det,
                          (b[3] * b[7] - b[4] * b[6]) / det, (b[1] * b[6] - b[0] * b[7]) / det, (b[0] * b[4] - b[1] * b[3]) / det };
        for (int64_t i = aoff[s]; i < aoff[s + 1]; ++i) {
            const double* r = pos + 3 * i;
            if (!std::isfinite(r[0]) || !std::isfinite(r[1]) || !std::isfinite(r[2])) return fail(c, NEP_EINVAL, "non-finite position");
            if (type[i] < 0 || type[i] >= c->m.T) return fail(c, NEP_EINVAL, "type out of range at atom " + std::to_string(i));
            for (int k = 0; k < 3; ++k) {
                double f = r[0] * inv[k] + r[1] * inv[3 + k] + r[2] * inv[6 + k];
                if (f < -1e-9 || f >= 1.0 + 1e-9)
                    return fail(c, NEP_EINVAL, "fractional coordinate outside [0,1) at atom " + std::to_string(i) + " (wrap positions first)");
            }
        }
    }
    free_dataset(c);
    c->S = S; c->N = N; c->NP = NP; c->nslices = (int)(NP / WARP);
    c->h_nat.assign(n_atoms, n_atoms + S); c->h_aoff = aoff; c->h_pbase = pbase; c->h_box.assign(box, box + 9 * (size_t)S);
    std::vector<int> slice_struct((size_t)c->nslices, 0);
    c->h_tcount.assign((size_t)S * c->m.T, 0);
    c->h_type.assign(type, type + N);
    c->h_slot_of.resize((size_t)N);
    c->h_Flab.clear();
    for (int s = 0; s < S; ++s) {
        for (int i = 0; i < n_atoms[s]; ++i) { c->h_slot_of[aoff[s] + i] = i; c->h_tcount[(size_t)s * c->m.T + type[aoff[s] + i]]++; }
        for (int64_t sl = pbase[s] / WARP; sl < pbase[s + 1] / WARP; ++sl) slice_struct[sl] = s;
    }
    DataDev& d = c->d;
    d.S = S; d.N = N; d.NP = NP; d.nslices = c->nslices;
    int rc;
    double *dpos, *dbox; int *dtype, *dss; int64_t *dao, *dpb;
    if ((rc = upload<double>(c, dpos, pos, 3 * (size_t)N))) return rc;
    if ((rc = upload<double>(c, dbox, box, 9 * (size_t)S))) return rc;
    if ((rc = upload<int>(c, dtype, type, (size_t)N))) return rc;
    if ((rc = upload<int>(c, dss, slice_struct.data(), slice_struct.size()))) return rc;
    if ((rc = upload<int64_t>(c, dao, aoff.data(), aoff.size()))) return rc;
    if ((rc = upload<int64_t>(c, dpb, pbase.data(), pbase.size()))) return rc;
    NEP_CUDA(c, cudaStreamSynchronize(c->stream));
    d.pos = dpos; d.box = dbox; d.type = dtype; d.slice_struct = dss; d.atom_off = dao; d.pbase = dpb;
    if ((rc = upload_slot_tables(c))) return rc;
    c->have_data = true;
    if (lab) return upload_labels(c, E, F, W, has_virial);
    c->h_hasv.assign(S, 1);
    return NEP_OK;
}

int nep_set_labels(nep_ctx* c, const double* E, const double* F, const double* W, const unsigned char* has_virial)
{
    CHECK_CTX(c);
    if (!c->have_data) return fail(c, NEP_ESTATE, "nep_set_labels before nep_load_structures");
    if (!E || !F || !W) return fail(c, NEP_EINVAL, "E, F and W are all required");
    int rc = upload_labels(c, E, F, W, has_virial);
    if (rc == NEP_OK && c->have_nbrs) {
        // S_v of the current batch depends on the mask.  All three normalisers of Eqs. 5-7 go back to the counts of the
        // local batch (as after nep_set_batch): a data-parallel caller gives the whole batch's counts again.
        int sv = 0;
        for (int sid : c->h_bsid) sv += c->h_hasv[sid];
        c->b.Sv = sv;
        c->b.nrmS = (double)c->b.Sb; c->b.nrmN = (double)c->b.Nb; c->b.nrmV = (double)sv;
        ++c->graph_gen;
    }
    return rc;
}

int nep_build_neighbors(nep_ctx* c)
{
    CHECK_CTX(c);
    if (!c->have_data) return fail(c, NEP_ESTATE, "nep_build_neighbors before nep_load_structures");
    c->batch_tables_valid = false;
    ++c->graph_gen;                            // the lists, the pair cache and the slot tables are released and allocated again: a captured
                                               // step graph holds the old pointers (StepArgs.d by value) whatever the batch tables look like
    int rc = build_neighbors_dev(c);
    if (rc) return rc;
    c->have_nbrs = true;
    return nep_set_batch(c, 0, nullptr);
}

int nep_get_neighbors(nep_ctx* c, int which, int64_t* n_pairs, int64_t* offsets, int* j, signed char* shift)
{
    CHECK_CTX(c);
    if (!c->have_nbrs) return fail(c, NEP_ESTATE, "nep_get_neighbors before nep_build_neighbors");
    if (which != 0 && which != 1) return fail(c, NEP_EINVAL, "which must be 0 (radial) or 1 (angular)");
    int64_t P = which ? c->PA : c->PR;
    if (n_pairs) *n_pairs = P;
    const DataDev& d = c->d;
    if (offsets) NEP_CUDA(c, cudaMemcpyAsync(offsets, which ? d.offA : d.offR, 8 * (size_t)(c->N + 1), cudaMemcpyDeviceToHost, c->stream));
    if (j && P) NEP_CUDA(c, cudaMemcpyAsync(j, which ? d.jA : d.jR, 4 * (size_t)P, cudaMemcpyDeviceToHost, c->stream));
    if (shift && P) NEP_CUDA(c, cudaMemcpyAsync(shift, which ? d.shA : d.shR, 3 * (size_t)P, cudaMemcpyDeviceToHost, c->stream));
    NEP_CUDA(c, cudaStreamSynchronize(c->stream));
    return NEP_OK;
}

static int h2d(nep_ctx* c, void* dst, const void* src, size_t bytes)
{
    NEP_CUDA(c, cudaMemcpyAsync(dst, src, bytes, cudaMemcpyHostToDevice, c->stream));
    NEP_CUDA(c, cudaStreamSynchronize(c->stream));
    return NEP_OK;
}
static int d2h(nep_ctx* c, void* dst, const void* src, size_t bytes)
{
    if (bytes <= sizeof c->h_small_bytes && c->h_small) {   // small results (the loss terms) through a pinned bounce buffer
        NEP_CUDA(c, cudaMemcpyAsync(c->h_small, src, bytes, cudaMemcpyDeviceToHost, c->stream));
        NEP_CUDA(c, cudaStreamSynchronize(c->stream));
        memcpy(dst, c->h_small, bytes);
        return NEP_OK;
    }
    NEP_CUDA(c, cudaMemcpyAsync(dst, src, bytes, cudaMemcpyDeviceToHost, c->stream));
    NEP_CUDA(c, cudaStreamSynchronize(c->stream));
    return NEP_OK;
}

int nep_set_params(nep_ctx* c, const float* theta)
{
    CHECK_CTX(c);
    if (!theta) return fail(c, NEP_EINVAL, "theta is NULL");
    for (int i = 0; i < c->m.npar; ++i) if (!std::isfinite(theta[i])) return fail(c, NEP_EINVAL, "non-finite parameter");
    c->have_params = true; c->forward_valid = c->grad_valid = false;
    return h2d(c, c->theta, theta, 4 * (size_t)c->m.npar);
}
int nep_get_params(nep_ctx* c, float* theta)
{
    CHECK_CTX(c);
    if (!theta) return fail(c, NEP_EINVAL, "theta is NULL");
    return d2h(c, theta, c->theta, 4 * (size_t)c->m.npar);
}
int nep_get_grad(nep_ctx* c, float* g)
{
    CHECK_CTX(c);
    if (!g) return fail(c, NEP_EINVAL, "g is NULL");
    if (!c->grad_valid) return fail(c, NEP_ESTATE, "no gradient: call nep_loss_grad (or nep_set_grad) first");
    return d2h(c, g, c->g, 4 * (size_t)c->m.npar);
}
// ---- a model as a file: hyper-parameters of Table I, the scaler of Eq. 2 and theta (layout DESIGN C0) ----
static const char* const MODEL_MAGIC = "nep_b200_model";
int nep_save_model(nep_ctx* c, const char* path)
{
    CHECK_CTX(c);
    if (!path) return fail(c, NEP_EINVAL, "path is NULL");
    if (!c->have_params || !c->have_scaler) return fail(c, NEP_ESTATE, "nep_save_model needs parameters and a scaler");
    std::vector<float> th(c->m.npar);
    std::vector<double> sc(c->m.D);
    int rc = nep_get_params(c, th.data());
    if (rc) return rc;
    if ((rc = nep_get_scaler(c, sc.data()))) return rc;
    FILE* f = fopen(path, "w");
    if (!f) return fail(c, NEP_EINVAL, std::string("cannot open ") + path + " for writing");
    fprintf(f, "%s 1\n", MODEL_MAGIC);
    fprintf(f, "n_species %d\ncutoff %.17g %.17g\nn_max %d %d\nbasis_size %d %d\nl_max %d %d %d\nneuron %d\n", c->m.T, c->rcR, c->rcA,
            c->n_max_R, c->n_max_A, c->basis_R, c->basis_A, c->l3, c->l4, c->l5, c->m.H);
    fprintf(f, "scaler %d\n", c->m.D);
    for (int i = 0; i < c->m.D; ++i) fprintf(f, "%.9g\n", sc[i]);          // the scaler is held in fp32 on the device
    fprintf(f, "theta %d\n", c->m.npar);
    for (int i = 0; i < c->m.npar; ++i) fprintf(f, "%.9g\n", th[i]);       // 9 significant digits round-trip an fp32 value
    const bool ok = !ferror(f);
    if (fclose(f) != 0 || !ok) return fail(c, NEP_EINVAL, std::string("write error on ") + path);
    return NEP_OK;
}
int nep_create_from_model_file(nep_ctx** out, const char* path, nep_alloc_fn alloc, nep_free_fn free_, void* alloc_user, void* cuda_stream)
{
    if (!out) return fail(nullptr, NEP_EINVAL, "out is NULL");
    *out = nullptr;
    if (!path) return fail(nullptr, NEP_EINVAL, "path is NULL");
    FILE* f = fopen(path, "r");
    if (!f) return fail(nullptr, NEP_EINVAL, std::string("cannot open ") + path);
    char magic[32] = {0};
    int ver = 0, T = 0, nmR = 0, nmA = 0, bR = 0, bA = 0, l3 = 0, l4 = 0, l5 = 0, H = 0, D = 0, npar = 0;
    double rcR = 0, rcA = 0;
    bool ok = fscanf(f, "%31s %d", magic, &ver) == 2 && std::string(magic) == MODEL_MAGIC && ver == 1;
    ok = ok && fscanf(f, " n_species %d cutoff %lf %lf n_max %d %d basis_size %d %d l_max %d %d %d neuron %d scaler %d", &T, &rcR, &rcA, &nmR,
                      &nmA, &bR, &bA, &l3, &l4, &l5, &H, &D) == 12;
    if (!ok) { fclose(f); return fail(nullptr, NEP_EINVAL, std::string(path) + " is not a nep_b200 model file (version 1)"); }
    nep_ctx* c = nullptr;
    int rc = nep_create(&c, T, rcR, rcA, nmR, nmA, bR, bA, l3, l4, l5, H, alloc, free_, alloc_user, cuda_stream);
    if (rc) { fclose(f); return rc; }
    std::vector<double> sc(c->m.D);
    std::vector<float> th(c->m.npar);
    ok = D == c->m.D;
    for (int i = 0; ok && i < D; ++i) ok = fscanf(f, "%lf", &sc[i]) == 1;
    ok = ok && fscanf(f, " theta %d", &npar) == 1 && npar == c->m.npar;
    for (int i = 0; ok && i < npar; ++i) ok = fscanf(f, "%f", &th[i]) == 1;
    fclose(f);
    if (!ok) { nep_destroy(c); return fail(nullptr, NEP_EINVAL, std::string(path) + ": sizes or values do not match the header"); }
    if ((rc = nep_set_params(c, th.data())) || (rc = nep_set_scaler(c, sc.data()))) {
        g_create_error = c->err;
        nep_destroy(c);
        return rc;
    }
    *out = c;
    return NEP_OK;
}
int nep_get_model(const nep_ctx* c, int* n_species, double* rc2, int* n_max2, int* basis2, int* l_max3, int* neurons)
{
    if (!c) return NEP_EINVAL;
    if (n_species) *n_species = c->m.T;
    if (rc2) { rc2[0] = c->rcR; rc2[1] = c->rcA; }
    if (n_max2) { n_max2[0] = c->n_max_R; n_max2[1] = c->n_max_A; }
    if (basis2) { basis2[0] = c->basis_R; basis2[1] = c->basis_A; }
    if (l_max3) { l_max3[0] = c->l3; l_max3[1] = c->l4; l_max3[2] = c->l5; }
    if (neurons) *neurons = c->m.H;
    return NEP_OK;
}
int nep_set_grad(nep_ctx* c, const float* g)
{
    CHECK_CTX(c);
    if (!g) return fail(c, NEP_EINVAL, "g is NULL");
    c->grad_valid = true;
    return h2d(c, c->g, g, 4 * (size_t)c->m.npar);
}
int nep_set_adam_state(nep_ctx* c, const float* m, const float* v, const float* vmax, int64_t t)
{
    CHECK_CTX(c);
    if (!m || !v || !vmax || t < 0) return fail(c, NEP_EINVAL, "bad Adam state");
    size_t nb = 4 * (size_t)c->m.npar;
    int rc;
    if ((rc = h2d(c, c->am, m, nb)) || (rc = h2d(c, c->av, v, nb)) || (rc = h2d(c, c->avmax, vmax, nb))) return rc;
    c->t_adam = t;
    return NEP_OK;
}
int nep_get_adam_state(nep_ctx* c, float* m, float* v, float* vmax, int64_t* t)
{
    CHECK_CTX(c);
    size_t nb = 4 * (size_t)c->m.npar;
    int rc;
    if (m && (rc = d2h(c, m, c->am, nb))) return rc;
    if (v && (rc = d2h(c, v, c->av, nb))) return rc;
    if (vmax && (rc = d2h(c, vmax, c->avmax, nb))) return rc;
    if (t) *t = c->t_adam;
    return NEP_OK;
}

int nep_set_scaler(nep_ctx* c, const double* s)
{
    CHECK_CTX(c);
    if (!s) return fail(c, NEP_EINVAL, "s is NULL");
    std::vector<float> f(c->m.DP, 0.0f);
    for (int i = 0; i < c->m.D; ++i) {
        if (!std::isfinite(s[i])) return fail(c, NEP_EINVAL, "non-finite scaler");
        f[i] = (float)s[i];
    }
    c->have_scaler = true; c->forward_valid = c->grad_valid = false;
    return h2d(c, c->scaler, f.data(), 4 * f.size());
}
int nep_get_scaler(nep_ctx* c, double* s)
{
    CHECK_CTX(c);
    if (!s) return fail(c, NEP_EINVAL, "s is NULL");
    if (!c->have_scaler) return fail(c, NEP_ESTATE, "no scaler yet");
    std::vector<float> f(c->m.DP);
    int rc = d2h(c, f.data(), c->scaler, 4 * f.size());
    if (rc) return rc;
    for (int i = 0; i < c->m.D; ++i) s[i] = f[i];
    return NEP_OK;
}
// descriptors of every loaded atom at the current parameters, then their per-component minimum and maximum (device)
static int descriptor_range_dev(nep_ctx* c, const char* who)
{
    if (!c->have_nbrs) return fail(c, NEP_ESTATE, std::string(who) + " before nep_build_neighbors");
    if (!c->have_params) return fail(c, NEP_ESTATE, std::string(who) + " before nep_set_params");
    int rc = nep_set_batch(c, 0, nullptr);
    if (rc) return rc;
    if (!c->qrange) { c->qrange = (float*)dev_alloc(c, 4 * 2 * (size_t)c->m.DP); if (!c->qrange) return NEP_ENOMEM; }
    if ((rc = launch_forward(c, true))) return rc;
    return launch_descriptor_range(c, c->qrange);
}
int nep_compute_scaler(nep_ctx* c)
{
    CHECK_CTX(c);
    int rc = descriptor_range_dev(c, "nep_compute_scaler");
    if (rc) return rc;
    if ((rc = launch_scaler_from_range(c, c->qrange, c->scaler))) return rc;
    NEP_CUDA(c, cudaStreamSynchronize(c->stream));
    c->have_scaler = true; c->forward_valid = c->grad_valid = false;
    return NEP_OK;
}
int nep_compute_descriptor_range(nep_ctx* c, double* qmin, double* qmax)
{
    CHECK_CTX(c);
    if (!qmin || !qmax) return fail(c, NEP_EINVAL, "qmin / qmax is NULL");
    int rc = descriptor_range_dev(c, "nep_compute_descriptor_range");
    if (rc) return rc;
    std::vector<float> f(2 * (size_t)c->m.DP);
    if ((rc = d2h(c, f.data(), c->qrange, 4 * f.size()))) return rc;
    for (int v = 0; v < c->m.D; ++v) { qmin[v] = f[v]; qmax[v] = f[c->m.DP + v]; }
    c->forward_valid = c->grad_valid = false;
    return NEP_OK;
}
int nep_set_scaler_from_range(nep_ctx* c, const double* qmin, const double* qmax)
{
    CHECK_CTX(c);
    if (!qmin || !qmax) return fail(c, NEP_EINVAL, "qmin / qmax is NULL");
    std::vector<float> f(2 * (size_t)c->m.DP, 0.0f);
    for (int v = 0; v < c->m.D; ++v) {
        if (std::isnan(qmin[v]) || std::isnan(qmax[v])) return fail(c, NEP_EINVAL, "NaN in descriptor range");
        f[v] = (float)qmin[v]; f[c->m.DP + v] = (float)qmax[v];
    }
    if (!c->qrange) { c->qrange = (float*)dev_alloc(c, 4 * f.size()); if (!c->qrange) return NEP_ENOMEM; }
    int rc = h2d(c, c->qrange, f.data(), 4 * f.size());
    if (rc) return rc;
    if ((rc = launch_scaler_from_range(c, c->qrange, c->scaler))) return rc;
    NEP_CUDA(c, cudaStreamSynchronize(c->stream));
    c->have_scaler = true; c->forward_valid = c->grad_valid = false;
    return NEP_OK;
}

static int ensure_batch_capacity(nep_ctx* c, int64_t NBP, int Sb, int nbs, int64_t tiles_m)
{
    BatchDev& b = c->b;
    const ModelDev& m = c->m;
    if (NBP > c->cap_NBP) {
        void* olds[] = { b.q, b.Fp, b.S, b.Sd, b.qd, b.Qb, b.arow, b.Bd, b.F, b.u, b.Ei };
        for (void* p : olds) dev_free(c, p);
        b.q = b.Fp = b.S = b.Sd = b.qd = b.Qb = b.arow = b.Bd = b.F = b.u = b.Ei = nullptr;   // a failed allocation below leaves no dangling pointer
        c->cap_NBP = 0;
        size_t n = (size_t)NBP;
        ALLOC(c, b.q, float, n * m.D);   ALLOC(c, b.Fp, float, n * m.D);
        ALLOC(c, b.S, float, n * m.nA * 24); ALLOC(c, b.Sd, float, n * m.nA * 24);
        ALLOC(c, b.qd, float, n * m.D);  ALLOC(c, b.Qb, float, n * m.D);
        ALLOC(c, b.arow, float, n * m.T * m.KRP); ALLOC(c, b.Bd, float, n * m.T * m.KR);
        ALLOC(c, b.F, float, n * 4);     ALLOC(c, b.u, float, n * 3);     ALLOC(c, b.Ei, float, n);
        c->cap_NBP = NBP;
    }
    if (tiles_m > c->cap_tiles_m) {
        dev_free(c, b.alist); dev_free(c, b.hbuf);
        b.alist = nullptr; b.hbuf = nullptr; c->cap_tiles_m = 0;
        ALLOC(c, b.alist, int, tiles_m);
        ALLOC(c, b.hbuf, float, (size_t)tiles_m * m.HP);
        c->cap_tiles_m = tiles_m;
    }
    if (Sb > c->cap_Sb) {
        void* olds[] = { b.Es, b.Ws, b.eps, b.G };
        for (void* p : olds) dev_free(c, p);
        b.Es = nullptr; b.Ws = b.eps = b.G = nullptr; c->cap_Sb = 0;
        ALLOC(c, b.Es, double, Sb); ALLOC(c, b.Ws, float, 9 * (size_t)Sb); ALLOC(c, b.eps, float, Sb); ALLOC(c, b.G, float, 9 * (size_t)Sb);
        c->cap_Sb = Sb;
    }
    if (!b.lacc) {   // loss accumulators and the block ticket: zero once, the loss kernel re-arms them itself
        ALLOC(c, b.lacc, double, 8 + 4 * 2 * (size_t)c->sm_count); ALLOC(c, b.counter, unsigned, 64);
        NEP_CUDA(c, cudaMemsetAsync(b.lacc, 0, 64, c->stream));
        NEP_CUDA(c, cudaMemsetAsync(b.counter, 0, 256, c->stream));
    }
    // per-batch tables: one pinned host block, one device block, one copy per nep_set_batch
    const size_t need = 16 * (size_t)nbs + 8 * (size_t)Sb + 4 * (size_t)Sb * (2 + m.T) + 64;
    if (need > c->d_stage_bytes) {
        NEP_CUDA(c, cudaStreamSynchronize(c->stream));   // no copy out of the old pinned block is pending
        dev_free(c, c->d_stage);
        if (c->h_stage) cudaFreeHost(c->h_stage);
        c->h_stage = nullptr; c->d_stage = nullptr; c->d_stage_bytes = 0;
        const size_t cap = need + need / 2;
        NEP_CUDA(c, cudaMallocHost(&c->h_stage, cap));
        c->d_stage = dev_alloc(c, cap);
        if (!c->d_stage) return NEP_ENOMEM;
        c->d_stage_bytes = c->h_stage_bytes = cap;
    }
    return NEP_OK;
}

int nep_set_batch(nep_ctx* c, int n, const int* ids)
{
    CHECK_CTX(c);
    if (!c->have_nbrs) return fail(c, NEP_ESTATE, "nep_set_batch before nep_build_neighbors");
    if (ids && n < 0) return fail(c, NEP_EINVAL, "negative batch size");
    const int Sb = ids ? n : c->S;
    const int T = c->m.T;
    // The same batch as the current one (full-batch training re-selects it every step): the tables in the pinned block and the
    // type-sorted atom list on the device are still those of this batch; only the upload is repeated.
    if (c->batch_tables_valid && Sb == c->b.Sb && Sb > 0 && (int)c->h_bsid.size() == Sb) {
        bool same = true;
        for (int k = 0; k < Sb && same; ++k) same = c->h_bsid[k] == (ids ? ids[k] : k);
        if (same) {
            const size_t bytes = 16 * (size_t)c->b.nbs + 8 * (size_t)Sb + 4 * (size_t)Sb * (2 + T);
            NEP_CUDA(c, cudaMemcpyAsync(c->d_stage, c->h_stage, bytes, cudaMemcpyHostToDevice, c->stream));
            c->forward_valid = c->grad_valid = false;
            const double nS = (double)c->b.Sb, nN = (double)c->b.Nb, nV = (double)c->b.Sv;              // as after any nep_set_batch
            if (c->b.nrmS != nS || c->b.nrmN != nN || c->b.nrmV != nV) ++c->graph_gen;
            c->b.nrmS = nS; c->b.nrmN = nN; c->b.nrmV = nV;
            return NEP_OK;
        }
    }
    c->batch_tables_valid = false;
    std::vector<unsigned char> seen(ids ? c->S : 0, 0);
    int64_t nbs64 = 0;
    for (int k = 0; k < Sb; ++k) {
        const int s = ids ? ids[k] : k;
        if (s < 0 || s >= c->S) return fail(c, NEP_EINVAL, "structure id out of range");
        if (ids) { if (seen[s]) return fail(c, NEP_EINVAL, "duplicate structure id in batch"); seen[s] = 1; }
        nbs64 += (c->h_pbase[s + 1] - c->h_pbase[s]) / WARP;
    }
    if (nbs64 * WARP > INT32_MAX / 2 || nbs64 * WARP * c->m.T * c->m.KRP > (int64_t)UINT32_MAX)
        return fail(c, NEP_ECAPACITY, "batch too large");   // 32-bit element indices into the per-atom rows
    const int nbs = (int)nbs64;
    // network tiles: atoms sorted by species, every species padded to whole tiles
    const int TM = ann_tile_m(c);
    std::vector<int64_t> tot(T, 0);
    for (int k = 0; k < Sb; ++k) {
        const int s = ids ? ids[k] : k;
        for (int t = 0; t < T; ++t) tot[t] += c->h_tcount[(size_t)s * T + t];
    }
    // a batch of the same shape in the same buffers leaves a captured step graph valid.  The snapshot is taken BEFORE the first tile
    // of each species is rewritten: StepArgs carries tile_start by value, so two batches that agree in every count but not in their
    // composition (other atoms per species) need a new capture.
    const BatchDev b_before = c->b;
    BatchDev& b = c->b;
    int ntiles = 0;
    for (int t = 0; t < T; ++t) { b.tile_start[t] = ntiles; ntiles += (int)((tot[t] + TM - 1) / TM); }
    for (int t = T; t <= MAX_T; ++t) b.tile_start[t] = ntiles;
    c->forward_valid = c->grad_valid = false;
    int rc = ensure_batch_capacity(c, std::max<int64_t>(nbs64 * WARP, WARP), std::max(Sb, 1), std::max(nbs, 1), std::max<int64_t>((int64_t)ntiles * TM, TM));
    if (rc) {   // no batch is selected after a failed allocation: the step calls launch nothing
        b.Sb = b.Sv = 0; b.Nb = 0; b.nbs = 0; b.NBP = 0; b.ntiles = 0;
        c->h_bsid.clear(); c->h_bfoff.clear();
        ++c->graph_gen;
        return rc;
    }
    // tables, packed: binfo [nbs] int4 | bfoff [Sb] int64 | bsid [Sb] | bnat [Sb] | bsoff [Sb][T]
    char* h = (char*)c->h_stage;
    int4* binfo = (int4*)h;
    int64_t* bfoff = (int64_t*)(h + 16 * (size_t)nbs);
    int* bsid = (int*)(bfoff + Sb);
    int* bnat = bsid + Sb;
    int* bsoff = bnat + Sb;
    NEP_CUDA(c, cudaStreamSynchronize(c->stream));   // the previous copy out of the pinned block has finished
    int64_t Nb = 0, nbp = 0, PRb = 0, PAb = 0;
    int Sv = 0, w = 0;
    std::vector<int> run(T, 0);
    for (int k = 0; k < Sb; ++k) {
        const int s = ids ? ids[k] : k;
        bsid[k] = s; bnat[k] = c->h_nat[s]; bfoff[k] = Nb;
        for (int t = 0; t < T; ++t) { bsoff[(size_t)k * T + t] = run[t]; run[t] += c->h_tcount[(size_t)s * T + t]; }
        Nb += c->h_nat[s];
        Sv += c->h_hasv.empty() ? 1 : c->h_hasv[s];
        PRb += c->h_pairsR_struct[s]; PAb += c->h_pairsA_struct[s];
        for (int64_t sl = c->h_pbase[s] / WARP; sl < c->h_pbase[s + 1] / WARP; ++sl) binfo[w++] = make_int4((int)sl, k, (int)nbp, 0);
        nbp += c->h_pbase[s + 1] - c->h_pbase[s];
    }
    b.Sb = Sb; b.Sv = Sv; b.Nb = Nb; b.nbs = nbs; b.NBP = nbp; b.tile_m = TM; b.ntiles = ntiles;
    b.nrmS = (double)Sb; b.nrmN = (double)Nb; b.nrmV = (double)Sv;
    const size_t bytes = 16 * (size_t)nbs + 8 * (size_t)Sb + 4 * (size_t)Sb * (2 + T);
    char* d = (char*)c->d_stage;
    b.binfo = (const int4*)d;
    b.bfoff = (const int64_t*)(d + 16 * (size_t)nbs);
    b.bsid = (const int*)(b.bfoff + Sb);
    b.bnat = b.bsid + Sb;
    b.bsoff = b.bnat + Sb;
    if (bytes) NEP_CUDA(c, cudaMemcpyAsync(c->d_stage, c->h_stage, bytes, cudaMemcpyHostToDevice, c->stream));
    c->h_bsid.assign(bsid, bsid + Sb); c->h_bfoff.assign(bfoff, bfoff + Sb); c->PRb = PRb; c->PAb = PAb;
    c->forward_valid = c->grad_valid = false;
    if (memcmp(&b_before, &c->b, sizeof(BatchDev)) != 0) ++c->graph_gen;
    rc = launch_build_alist(c);
    c->batch_tables_valid = rc == NEP_OK;
    return rc;
}

static int copy_out(nep_ctx* c, void* dst, const float* src, size_t count, int on_host)
{
    if (!dst || !count) return NEP_OK;
    NEP_CUDA(c, cudaMemcpyAsync(dst, src, 4 * count, on_host ? cudaMemcpyDeviceToHost : cudaMemcpyDeviceToDevice, c->stream));
    return NEP_OK;
}

int nep_forward(nep_ctx* c, void* E_out, void* F_out, void* W_out, int on_host)
{
    CHECK_CTX(c);
    if (!c->have_nbrs) return fail(c, NEP_ESTATE, "nep_forward before nep_build_neighbors");
    if (!c->have_params) return fail(c, NEP_ESTATE, "nep_forward before nep_set_params");
    if (!c->have_scaler) return fail(c, NEP_ESTATE, "nep_forward before nep_set_scaler / nep_compute_scaler");
    int rc = launch_forward(c, false);
    if (rc) return rc;
    c->forward_valid = true; c->grad_valid = false; c->loss_valid = false;
    if (E_out || F_out || W_out) {
        const BatchDev& b = c->b;
        size_t nE = (size_t)b.Sb, nF = 3 * (size_t)b.Nb, nW = 9 * (size_t)b.Sb;
        if (on_host) {
            float* stage = (float*)dev_alloc(c, 4 * (nE + nF + nW + 1));
            if (!stage) return NEP_ENOMEM;
            rc = launch_gather_outputs(c, E_out ? stage : nullptr, F_out ? stage + nE : nullptr, W_out ? stage + nE + nF : nullptr);
            if (!rc) rc = copy_out(c, E_out, stage, nE, 1);
            if (!rc) rc = copy_out(c, F_out, stage + nE, nF, 1);
            if (!rc) rc = copy_out(c, W_out, stage + nE + nF, nW, 1);
            cudaError_t e = cudaStreamSynchronize(c->stream);
            dev_free(c, stage);
            if (rc) return rc;
            if (e != cudaSuccess) return fail(c, NEP_ECUDA, std::string("nep_forward: ") + cudaGetErrorString(e));
        } else {
            if ((rc = launch_gather_outputs(c, (float*)E_out, (float*)F_out, (float*)W_out))) return rc;
        }
    }
    return NEP_OK;
}

int nep_get_descriptors(nep_ctx* c, float* q)
{
    CHECK_CTX(c);
    if (!q) return fail(c, NEP_EINVAL, "q is NULL");
    if (!c->forward_valid) return fail(c, NEP_ESTATE, "nep_get_descriptors needs nep_forward first");
    size_t n = (size_t)c->b.Nb * c->m.D;
    float* stage = (float*)dev_alloc(c, 4 * std::max<size_t>(n, 1));
    if (!stage) return NEP_ENOMEM;
    int rc = launch_gather_q(c, stage);
    if (!rc) rc = d2h(c, q, stage, 4 * n);
    dev_free(c, stage);
    return rc;
}

int nep_set_batch_normalisers(nep_ctx* c, int64_t n_struct, int64_t n_atoms, int64_t n_virial)
{
    CHECK_CTX(c);
    if (!c->have_nbrs) return fail(c, NEP_ESTATE, "nep_set_batch_normalisers before nep_build_neighbors");
    if (n_struct < c->b.Sb || n_atoms < c->b.Nb || n_virial < c->b.Sv)
        return fail(c, NEP_EINVAL, "the whole batch cannot be smaller than this context's share of it");
    c->b.nrmS = (double)n_struct; c->b.nrmN = (double)n_atoms; c->b.nrmV = (double)n_virial;
    c->grad_valid = false;
    ++c->graph_gen;
    return NEP_OK;
}

int nep_grad_device_ptr(nep_ctx* c, float** g, double** loss4)
{
    CHECK_CTX(c);
    if (!c->b.lacc) return fail(c, NEP_ESTATE, "nep_grad_device_ptr before nep_build_neighbors");
    if (g) *g = c->g;
    if (loss4) *loss4 = c->b.lacc + 4;
    return NEP_OK;
}

int nep_get_loss(nep_ctx* c, double* loss4)
{
    CHECK_CTX(c);
    if (!loss4) return fail(c, NEP_EINVAL, "loss4 is NULL");
    if (!c->loss_valid) return fail(c, NEP_ESTATE, "nep_get_loss needs nep_loss_grad first");
    return d2h(c, loss4, c->b.lacc + 4, 32);
}

int nep_loss_grad(nep_ctx* c, double lambda_E, double lambda_F, double lambda_V, double* loss4_host)
{
    CHECK_CTX(c);
    if (!c->forward_valid) return fail(c, NEP_ESTATE, "nep_loss_grad needs nep_forward on the same batch and parameters first");
    if (!c->have_labels) return fail(c, NEP_ESTATE, "nep_loss_grad needs labels (nep_load_structures / nep_set_labels)");
    if (!(lambda_E >= 0) || !(lambda_F >= 0) || !(lambda_V >= 0)) return fail(c, NEP_EINVAL, "loss weights must be >= 0");
    c->lamE = lambda_E; c->lamF = lambda_F; c->lamV = lambda_V;
    int rc = launch_loss_grad(c);
    if (rc) return rc;
    c->grad_valid = true; c->loss_valid = true;
    if (loss4_host) return d2h(c, loss4_host, c->b.lacc + 4, 32);
    return NEP_OK;
}

int nep_adam_step(nep_ctx* c, double lr, double beta1, double beta2, double eps, int variant)
{
    CHECK_CTX(c);
    if (!c->grad_valid) return fail(c, NEP_ESTATE, "nep_adam_step needs a gradient (nep_loss_grad)");
    if (!(lr >= 0) || !(beta1 >= 0 && beta1 < 1) || !(beta2 >= 0 && beta2 < 1) || !(eps >= 0) || (variant != 0 && variant != 1))
        return fail(c, NEP_EINVAL, "bad Adam hyper-parameter");
    int rc = launch_adam(c, lr, beta1, beta2, eps, variant);
    if (rc) return rc;
    c->forward_valid = false; c->grad_valid = false;
    return NEP_OK;
}

int nep_synchronize(nep_ctx* c)
{
    CHECK_CTX(c);
    NEP_CUDA(c, cudaStreamSynchronize(c->stream));
    return NEP_OK;
}

int nep_launch_count(nep_ctx* c, int64_t* n)
{
    CHECK_CTX(c);
    if (n) *n = c->launches;
    return NEP_OK;
}
int nep_profile_enable(nep_ctx* c, int on)
{
    CHECK_CTX(c);
    cudaStreamSynchronize(c->stream);
    for (auto& r : c->prof.pending) { c->prof.pool.push_back(r.a); c->prof.pool.push_back(r.b); }
    c->prof.pending.clear(); c->prof.acc.clear();
    c->prof.on = on != 0; c->prof.paused = false;
    return NEP_OK;
}
int nep_profile_pause(nep_ctx* c, int paused)
{
    CHECK_CTX(c);
    c->prof.paused = paused != 0;
    return NEP_OK;
}
int nep_profile_read(nep_ctx* c, int cap, const char** names, double* ms, int64_t* launches, int* n)
{
    CHECK_CTX(c);
    NEP_CUDA(c, cudaStreamSynchronize(c->stream));
    static thread_local std::vector<std::string> keep;
    for (auto& r : c->prof.pending) {
        float t = 0.f;
        cudaEventElapsedTime(&t, r.a, r.b);
        auto& a = c->prof.acc[r.name];
        a.first += t; a.second += 1;
        c->prof.pool.push_back(r.a); c->prof.pool.push_back(r.b);
    }
    c->prof.pending.clear();
    keep.clear();
    int k = 0;
    for (auto& kv : c->prof.acc) keep.push_back(kv.first);
    for (auto& kv : c->prof.acc) {
        if (k >= cap) break;
        if (names) names[k] = keep[k].c_str();
        if (ms) ms[k] = kv.second.first;
        if (launches) launches[k] = kv.second.second;
        ++k;
    }
    if (n) *n = k;
    c->prof.acc.clear();
    return NEP_OK;
}

int nep_network_on_tensor_cores(const nep_ctx* c) { return c && c->ann_tc ? 1 : 0; }

int nep_get_sizes(nep_ctx* c, int64_t* s)
{
    CHECK_CTX(c);
    if (!s) return fail(c, NEP_EINVAL, "sizes8 is NULL");
    s[0] = c->S; s[1] = c->N; s[2] = c->PR; s[3] = c->PA; s[4] = c->b.Sb; s[5] = c->b.Nb; s[6] = c->PRb; s[7] = c->PAb;
    return NEP_OK;
}

}  // extern "C"
