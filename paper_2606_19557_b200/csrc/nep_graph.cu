// nep_graph.cu -- one training step as ONE CUDA graph launch ("capturable as one CUDA graph").
//
// nep_train_step = nep_forward + nep_loss_grad + nep_adam_step on the current batch.  With use_graph the ten kernels are
// captured once from the context's stream (the same launchers the three calls use) and replayed with cudaGraphLaunch; the
// arguments that change from step to step -- the loss weights of Eq. 4, the learning rate and the bias corrections of
// Eqs. 11 -- are written into the nodes of k_loss and k_adam before every launch (cudaGraphExecKernelNodeSetParams), so the
// graph survives the learning-rate schedule and the two-stage protocol.  Everything that changes pointers or launch shapes
// (nep_set_batch, nep_set_batch_normalisers, labels, a new data set) bumps c->graph_gen and the step is captured again.
#include "nep_kernels.cuh"

namespace nep {

void graph_drop(nep_ctx* c)
{
    if (c->graph_exec) { cudaGraphExecDestroy(c->graph_exec); c->graph_exec = nullptr; }
    if (c->graph) { cudaGraphDestroy(c->graph); c->graph = nullptr; }
    c->graph_loss_node = nullptr; c->graph_adam_node = nullptr;
}

static int capture_step(nep_ctx* c, double lr, double b1, double b2, double eps, int variant)
{
    graph_drop(c);
    // captured from a stream of its own (the caller's may be the legacy default stream, which cannot be captured); the
    // launchers enqueue on c->stream, so it points there for the duration of the capture
    if (!c->cap_stream) NEP_CUDA(c, cudaStreamCreateWithFlags(&c->cap_stream, cudaStreamNonBlocking));
    cudaStream_t user_stream = c->stream;
    NEP_CUDA(c, cudaStreamBeginCapture(c->cap_stream, cudaStreamCaptureModeThreadLocal));
    c->stream = c->cap_stream;
    const int64_t t_before = c->t_adam, launches_before = c->launches;
    const bool prof_paused = c->prof.paused;
    c->prof.paused = true;                                  // no event records inside a capture
    c->capturing = true;
    int rc = launch_forward(c, false);
    if (!rc) rc = launch_loss_grad(c);
    if (!rc) rc = launch_adam(c, lr, b1, b2, eps, variant);
    c->capturing = false;
    c->prof.paused = prof_paused;
    c->t_adam = t_before;                                   // capturing is not stepping
    c->graph_launches = (int)(c->launches - launches_before);
    c->launches = launches_before;
    c->stream = user_stream;
    cudaGraph_t g = nullptr;
    cudaError_t e = cudaStreamEndCapture(c->cap_stream, &g);
    if (rc) { if (g) cudaGraphDestroy(g); return rc; }
    NEP_CUDA(c, e);
    c->graph = g;
    NEP_CUDA(c, cudaGraphInstantiate(&c->graph_exec, g, 0));
    size_t n = 0;
    NEP_CUDA(c, cudaGraphGetNodes(g, nullptr, &n));
    std::vector<cudaGraphNode_t> nodes(n);
    NEP_CUDA(c, cudaGraphGetNodes(g, nodes.data(), &n));
    LossArgs L; AdamArgs A;
    loss_args(c, make_args(c), &L);
    adam_args(c, lr, b1, b2, eps, variant, 1, &A);
    for (cudaGraphNode_t nd : nodes) {
        cudaGraphNodeType ty;
        NEP_CUDA(c, cudaGraphNodeGetType(nd, &ty));
        if (ty != cudaGraphNodeTypeKernel) continue;
        cudaKernelNodeParams p;
        NEP_CUDA(c, cudaGraphKernelNodeGetParams(nd, &p));
        if (p.func == L.func) { c->graph_loss_node = nd; c->graph_loss_grid = p.gridDim.x; }
        if (p.func == A.func) { c->graph_adam_node = nd; c->graph_adam_grid = p.gridDim.x; }
    }
    if (!c->graph_loss_node || !c->graph_adam_node) { graph_drop(c); return fail(c, NEP_ECUDA, "step graph: loss / Adam node not found"); }
    c->graph_built_gen = c->graph_gen; c->graph_variant = variant;
    return NEP_OK;
}

}  // namespace nep

using namespace nep;

extern "C" int nep_train_step(nep_ctx* c, double lambda_E, double lambda_F, double lambda_V, double lr, double beta1, double beta2,
                              double eps, int variant, int use_graph)
{
    if (!c) return NEP_EINVAL;
    if (!c->have_nbrs || !c->have_params || !c->have_scaler) return fail(c, NEP_ESTATE, "nep_train_step needs neighbours, parameters and a scaler");
    if (!c->have_labels) return fail(c, NEP_ESTATE, "nep_train_step needs labels (nep_load_structures / nep_set_labels)");
    if (!(lambda_E >= 0) || !(lambda_F >= 0) || !(lambda_V >= 0)) return fail(c, NEP_EINVAL, "loss weights must be >= 0");
    if (!(lr >= 0) || !(beta1 >= 0 && beta1 < 1) || !(beta2 >= 0 && beta2 < 1) || !(eps >= 0) || (variant != 0 && variant != 1))
        return fail(c, NEP_EINVAL, "bad Adam hyper-parameter");
    c->lamE = lambda_E; c->lamF = lambda_F; c->lamV = lambda_V;
    int rc;
    // a batch that is used once is not worth a capture (about a step's time on the host): the first step after anything that
    // invalidates the graph runs as three calls, the graph is captured when the same batch comes a second time
    const bool repeat = c->graph_seen_gen == c->graph_gen;
    c->graph_seen_gen = c->graph_gen;
    if (!use_graph || !repeat || c->b.nbs == 0) {
        if ((rc = launch_forward(c, false)) || (rc = launch_loss_grad(c)) || (rc = launch_adam(c, lr, beta1, beta2, eps, variant))) return rc;
    } else {
        if (!c->graph_exec || c->graph_built_gen != c->graph_gen || c->graph_variant != variant)
            if ((rc = capture_step(c, lr, beta1, beta2, eps, variant))) return rc;
        c->t_adam += 1;
        LossArgs L; AdamArgs A;
        loss_args(c, make_args(c), &L);
        adam_args(c, lr, beta1, beta2, eps, variant, c->t_adam, &A);
        cudaKernelNodeParams p{};
        p.func = const_cast<void*>(L.func); p.gridDim = dim3(c->graph_loss_grid); p.blockDim = dim3(256); p.sharedMemBytes = 0; p.kernelParams = L.ptrs; p.extra = nullptr;
        NEP_CUDA(c, cudaGraphExecKernelNodeSetParams(c->graph_exec, c->graph_loss_node, &p));
        p.func = const_cast<void*>(A.func); p.gridDim = dim3(c->graph_adam_grid); p.kernelParams = A.ptrs;
        NEP_CUDA(c, cudaGraphExecKernelNodeSetParams(c->graph_exec, c->graph_adam_node, &p));
        NEP_CUDA(c, cudaGraphLaunch(c->graph_exec, c->stream));
        c->launches += c->graph_launches;
    }
    c->forward_valid = false; c->grad_valid = false; c->loss_valid = true;
    return NEP_OK;
}
