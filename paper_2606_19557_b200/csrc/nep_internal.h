// nep_internal.h -- context, device views and launcher declarations shared by the .cu files of libnep_b200.
//
// Data layout.  Atoms of a structure are cut into SLICES of 32 (one warp = one slice, one
// lane = one atom, the last slice of a structure padded).  Every per-atom array the pair sweeps touch is
// "slice-blocked": element (slice w, row r, lane l) lives at ((w * ROWS) + r) * 32 + l, so a warp reads or writes
// 128 contiguous bytes per row and the row offset is an immediate in the instruction.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <map>
#include <string>
#include <vector>

#include "../../include/nep.h"

namespace nep {

constexpr int WARP = 32;
constexpr int MAX_T = 16;
constexpr int MAX_NCH = 5;   // angular channels held in registers by one thread

// Everything a kernel needs to know about the model (passed by value).
struct ModelDev {
    int T, nR, nA, KR, KA, KRP, H, HP, D, DP, nang, l3, has4, has5;   // HP, DP: H, D padded to multiples of 8; KRP: KR to 4; l3: 3-body orders l = 1..l3
    float rcR, rcA, rcinvR, rcinvA;
    // offsets into theta
    int per_type;          // (D + 2) * H
    int o_b1, o_cR, o_cA;
    int npar;
};

// Resident data set (positions fixed for the whole training run).
struct DataDev {
    int S;                 // structures
    int64_t N;             // atoms
    int64_t NP;            // padded atoms: every structure padded to a multiple of 32
    int nslices;           // NP / 32
    const double* pos;     // [N][3]
    const double* box;     // [S][9]
    const int* type;       // [N]
    const int64_t* atom_off;   // [S+1]
    const int64_t* pbase;      // [S+1] padded offset of each structure
    const int* type_p;     // [NP], -1 = padding
    const int* orig_p;     // [NP] structure-local index (caller's order) of the atom in this slot, -1 = padding
    const int* slot_of;    // [N]  structure-local slot of every atom: the inverse of orig_p
    const int* rank_p;     // [NP] rank of the atom among the atoms of its own type in its structure
    const int* slice_struct;   // [nslices]
    // labels
    const double* Elab;    // [S]
    const float* Flab;     // [nslices][3][32]
    const float* Wlab;     // [S][9]
    const unsigned char* hasv; // [S]
    // canonical neighbour lists (CSR over the N atoms)
    const int64_t* offR; const int* jR; const signed char* shR;
    const int64_t* offA; const int* jA; const signed char* shA;
    // sliced pair cache: record (slice, slot s, lane) at rec[recoff[slice] + s*32 + lane]
    const int* cntR; const int64_t* recoffR; const float4* recR;
    const int* cntA; const int64_t* recoffA; const float4* recA;
    const int* cntH; const int64_t* recoffH; const float4* recH;   // half list of the radial pairs (one record per undirected pair; nep_neighbor.cu)
    const float* B;        // [nslices][T*KR][32] radial aggregate  B_k[T'] = sum_{j in N_R(i), t_j = T'} f_k(r_ij)
};

// Current mini-batch: a list of slices; per-step temporaries are slice-blocked over the batch slices.
struct BatchDev {
    int Sb;                // structures in the batch
    int Sv;                // ... of which have virial labels
    int64_t Nb;            // atoms in the batch
    double nrmS, nrmN, nrmV;   // normalisers of Eqs. 5-7: S_b, N_b, S_v of the WHOLE batch (= the local ones unless data-parallel)
    int nbs;               // slices in the batch
    int64_t NBP;           // nbs * 32
    const int4* binfo;     // [nbs] {data-set slice, batch structure index, batch-padded index of the structure's first atom, 0}
    const int* bsid;       // [Sb]  data-set structure id
    const int* bnat;       // [Sb]  atoms of the structure
    const int64_t* bfoff;  // [Sb]  first atom in batch order (unpadded), for outputs
    const int* bsoff;      // [Sb][T] atoms of type t in the earlier structures of the batch
    // network tiles: atoms of the batch sorted by type, each type padded to a multiple of the tile size
    int tile_m;            // atoms per tile (128 or 64)
    int ntiles;
    int tile_start[MAX_T + 1];   // first tile of each type
    int* alist;            // [ntiles * tile_m] batch-padded atom index, -1 = padding
    // temporaries
    float* q;      // [nbs][D][32]   unscaled descriptors
    float* Fp;     // [nbs][D][32]   dE_i/dq
    float* qd;     // [nbs][D][32]   tangent of q (angular rows; radial rows are formed inside the network kernel)
    float* Qb;     // [nbs][D][32]   adjoint of q
    float* S;      // [nbs][nA*24][32] normalised angular moments
    float* Sd;     // [nbs][nA*24][32] their tangent
    float* hbuf;   // [ntiles][HP][tile_m] tanh outputs, tile order
    float* arow;   // [NBP][T*KRP]   a_k[T'] = sum_n Fp_n cR[t_i][T'][n][k]
    float* Bd;     // [nbs][T*KR][32] tangent of B
    float* F;      // [NBP][4]  (F_x, F_y, F_z, unused) per batch-padded atom: one 16-byte cell, scattered to with vector REDs
    float* u;      // [nbs][3][32]   dL/dF
    float* Ei;     // [nbs][32]
    // per structure
    double* Es;    // [Sb]
    float* Ws;     // [Sb][9]
    float* eps;    // [Sb]       dL/dE_s
    float* G;      // [Sb][9]    dL/dW_s
    double* lacc;  // loss4 = {L, dE, dF, dV} at [4..7]; [8 + 4 b ..]: partial sums (dE)^2, |dF|^2, (dW)^2, sum eps N of block b of the loss kernel
    unsigned* counter;   // [64] [0]: block ticket of the loss kernel
};

// Short-range pair correction (DESIGN G29): phi_ij(r) = sw(r) pref[ti][tj] / r sum_m coef_m exp(-expo_m r ainv[ti][tj]).
// Every number is the caller's (nep_set_pair_correction); passed to the kernel by value.
constexpr int MAX_PAIR_TERMS = 8;
struct PairCorrDev {
    int n_terms;
    float r_inner, r_outer, inv_width;       // inv_width = 1 / (r_outer - r_inner)
    float coef[MAX_PAIR_TERMS], expo[MAX_PAIR_TERMS];
    float pref[MAX_T * MAX_T];               // k_C Z_i Z_j
    float ainv[MAX_T * MAX_T];               // (Z_i^p + Z_j^p) / a_prefac
};

struct Profiler {
    bool on = false;
    bool paused = false;   // events are skipped while paused (the accumulators are kept)
    struct Rec { cudaEvent_t a, b; const char* name; };
    std::vector<Rec> pending;
    std::map<std::string, std::pair<double, int64_t>> acc;
    std::vector<cudaEvent_t> pool;
};

}  // namespace nep

struct nep_ctx {
    nep::ModelDev m;
    double rcR, rcA;
    int n_max_R, n_max_A, basis_R, basis_A, l3, l4, l5;
    nep_alloc_fn alloc; nep_free_fn free_; void* user;
    cudaStream_t stream;
    std::string err;
    std::vector<void*> allocs;
    int sm_count; int max_smem_optin; int max_smem_sm;
    bool ann_tc = false;   // network kernels on tcgen05 (nep_ann_tc.cu) instead of the FFMA tiles (nep_ann.cu)

    // host copies of the data set
    int S = 0; int64_t N = 0, NP = 0; int nslices = 0;
    std::vector<int> h_nat; std::vector<int64_t> h_aoff, h_pbase; std::vector<unsigned char> h_hasv;
    std::vector<int> h_tcount;   // [S][T] atoms of each type
    std::vector<double> h_box;
    // Slot order inside a structure: atoms sorted by (species, angular neighbour count) so that the
    // 32 lanes of a slice share a species and walk pair lists of similar length.  Identity until the lists exist.
    std::vector<int> h_type, h_slot_of;   // [N] species ; structure-local slot of every atom
    std::vector<float> h_Flab;            // [N][3] force labels in the caller's order (re-laid out when the slot order changes)
    bool have_data = false, have_labels = false, have_nbrs = false, have_params = false, have_scaler = false;
    bool forward_valid = false, grad_valid = false, loss_valid = false;   // loss_valid: the loss terms of the last nep_loss_grad are still on the device
    int64_t PR = 0, PA = 0;

    nep::DataDev d{};
    nep::BatchDev b{};
    int64_t cap_NBP = 0; int cap_Sb = 0; int cap_nbs = 0; int64_t cap_tiles_m = 0;
    std::vector<int> h_bsid; std::vector<int64_t> h_bfoff;
    bool batch_tables_valid = false;   // the pinned block and the device tables hold the tables of batch h_bsid (nep_set_batch fast path)
    int64_t PRb = 0, PAb = 0;
    std::vector<int64_t> h_pairsR_struct, h_pairsA_struct;   // pairs per structure (for sizes / flop models)
    // pinned staging for the per-batch tables (one async copy per nep_set_batch)
    void* h_stage = nullptr; size_t h_stage_bytes = 0; void* d_stage = nullptr; size_t d_stage_bytes = 0;
    void* h_small = nullptr; char h_small_bytes[64];   // pinned bounce buffer (and its size) for small device -> host results

    float *theta = nullptr, *g = nullptr, *am = nullptr, *av = nullptr, *avmax = nullptr, *scaler = nullptr;
    float* qrange = nullptr;   // [2][DP] per-component minimum and maximum of the descriptors (S0c)
    int64_t t_adam = 0;
    double lamE = 0, lamF = 0, lamV = 0;

    int64_t launches = 0;
    nep::Profiler prof;
    bool pair_on = false; nep::PairCorrDev pair{};   // short-range pair correction added to E, F, W by nep_forward (nep_pair.cu)

    // one training step as a CUDA graph (nep_graph.cu); graph_gen is bumped by every call that changes pointers or launch shapes
    cudaGraph_t graph = nullptr; cudaGraphExec_t graph_exec = nullptr; cudaStream_t cap_stream = nullptr;
    // small batches: the independent radial / angular sweeps of a step are captured as parallel branches (nep_misc.cu: SweepFork)
    bool capturing = false; cudaStream_t side_stream = nullptr; cudaEvent_t ev_fork = nullptr, ev_join = nullptr;
    cudaGraphNode_t graph_loss_node = nullptr, graph_adam_node = nullptr;
    unsigned graph_loss_grid = 0, graph_adam_grid = 0;
    int64_t graph_gen = 0, graph_built_gen = -1, graph_seen_gen = -1;
    int graph_variant = 0, graph_launches = 0;
};

namespace nep {

// ---- helpers implemented in nep_api.cu ----
int fail(nep_ctx* c, int code, const std::string& msg);
void* dev_alloc(nep_ctx* c, size_t bytes);        // nullptr on failure (err set)
void dev_free(nep_ctx* c, void* p);
void prof_begin(nep_ctx* c, const char* name);
void prof_end(nep_ctx* c);

#define NEP_CUDA(c, expr)                                                                     \
    do {                                                                                      \
        cudaError_t e__ = (expr);                                                             \
        if (e__ != cudaSuccess)                                                               \
            return nep::fail((c), NEP_ECUDA, std::string(#expr) + ": " + cudaGetErrorString(e__)); \
    } while (0)

// ---- launchers (each returns NEP_OK or an error code with c->err set) ----
int upload_slot_tables(nep_ctx* c);                            // nep_api.cu      : type_p, rank_p, orig_p, slot_of, force labels from h_slot_of
int build_neighbors_dev(nep_ctx* c);                           // nep_neighbor.cu : S0a + S0b
int launch_forward(nep_ctx* c, bool descriptors_only);         // nep_misc.cu     : S1-S5
int launch_loss_grad(nep_ctx* c);                              // nep_misc.cu     : S6-S9
int launch_adam(nep_ctx* c, double lr, double b1, double b2, double eps, int variant);  // nep_adam.cu : S10
int launch_descriptor_range(nep_ctx* c, float* d_rng);         // nep_misc.cu     : S0c min / max of q (after a descriptors-only pass over all)
int launch_scaler_from_range(nep_ctx* c, const float* d_rng, float* d_s);   //         : S0c s = 1 / (max - min)
int launch_gather_outputs(nep_ctx* c, float* dE, float* dF, float* dW);  // nep_misc.cu: slice-blocked -> batch order
int launch_gather_q(nep_ctx* c, float* dq);                    // [N_b][D]
int launch_build_alist(nep_ctx* c);                            // nep_misc.cu     : type-sorted atom list of the batch
int launch_pair_correction(nep_ctx* c);                        // nep_pair.cu     : short-range pair term added to E_s, F, W_s (after the force sweeps)
void graph_drop(nep_ctx* c);                                   // nep_graph.cu    : releases the captured step graph
int ann_tile_m(const nep_ctx* c);                              // nep_ann.cu      : atoms per network tile for this model

}  // namespace nep
