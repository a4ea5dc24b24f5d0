// hr_host.cu — host-buffer entry points with the gauge field resident on the device (include/hr_dslash.h, "host path").
// The gauge field changes once per molecular-dynamics step, the operator is applied hundreds of times in between
// ("recomputed whenever the gauge field is updated"): hr_gauge_upload_host moves the links once, and
// hr_apply_host_batch streams right-hand sides through the device in a three-stage pipeline — upload of spinor i+1,
// pack/operator/unpack of spinor i, download of result i-1 — so that both PCIe directions are busy at the same time.
#include <cstring>
#include <mutex>

#include "hr_common.cuh"

namespace hr {

static size_t up256h(size_t n) { return (n + 255) & ~(size_t)255; }

// two copy streams and the events of the pipeline, per device, created on first use and kept for the process
struct HostPipe {
    cudaStream_t s_in = nullptr, s_out = nullptr;
    cudaEvent_t start = nullptr, in[2] = {}, packed[2] = {}, out[2] = {}, done[2] = {};
    bool ready = false;
};
static HostPipe g_pipes[64];
static std::mutex g_pipe_mutex;

static int pipe_for_current_device(HostPipe** p) {
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 64) { set_error("host path: no usable CUDA device"); return HR_ECUDA; }
    std::lock_guard<std::mutex> lock(g_pipe_mutex);
    HostPipe& q = g_pipes[dev];
    if (!q.ready) {
        cudaError_t e = cudaStreamCreateWithFlags(&q.s_in, cudaStreamNonBlocking);
        if (e == cudaSuccess) e = cudaStreamCreateWithFlags(&q.s_out, cudaStreamNonBlocking);
        if (e == cudaSuccess) e = cudaEventCreateWithFlags(&q.start, cudaEventDisableTiming);
        for (int b = 0; b < 2 && e == cudaSuccess; ++b) {
            e = cudaEventCreateWithFlags(&q.in[b], cudaEventDisableTiming);
            if (e == cudaSuccess) e = cudaEventCreateWithFlags(&q.packed[b], cudaEventDisableTiming);
            if (e == cudaSuccess) e = cudaEventCreateWithFlags(&q.out[b], cudaEventDisableTiming);
            if (e == cudaSuccess) e = cudaEventCreateWithFlags(&q.done[b], cudaEventDisableTiming);
        }
        if (e != cudaSuccess) { set_error("host path: creating streams/events: %s", cudaGetErrorString(e)); return HR_ECUDA; }
        q.ready = true;
    }
    *p = &q;
    return HR_OK;
}

}  // namespace hr

using namespace hr;

#define HR_TRY(expr)                  \
    do {                              \
        int rc_ = (expr);             \
        if (rc_ != HR_OK) return rc_; \
    } while (0)
#define HR_CUDA(call)                                                                                       \
    do {                                                                                                    \
        cudaError_t e_ = (call);                                                                            \
        if (e_ != cudaSuccess) { set_error("%s: %s", #call, cudaGetErrorString(e_)); return HR_ECUDA; }     \
    } while (0)

extern "C" {

int hr_gauge_upload_host(const hr_geom* g, int rep, const void* u_canon_host, void* u_dev, void* workspace, void* stream) {
    if (!g || !u_canon_host) { set_error("hr_gauge_upload_host: NULL argument"); return HR_EINVAL; }
    const size_t cg = hr_canonical_gauge_bytes(g, rep);
    if (cg == 0) { set_error("hr_gauge_upload_host: invalid geometry or representation"); return HR_EINVAL; }
    if (!u_dev || !workspace || ((uintptr_t)u_dev & 15) || ((uintptr_t)workspace & 15)) { set_error("hr_gauge_upload_host: u_dev / workspace NULL or not 16-byte aligned"); return HR_EINVAL; }
    cudaStream_t st = (cudaStream_t)stream;
    HR_CUDA(cudaMemcpyAsync(workspace, u_canon_host, cg, cudaMemcpyHostToDevice, st));
    HR_TRY(hr_pack_gauge(g, rep, workspace, u_dev, stream));
    HR_CUDA(cudaStreamSynchronize(st));
    return HR_OK;
}

size_t hr_host_batch_workspace_bytes(const hr_geom* g) {
    const size_t cs = hr_canonical_spinor_bytes(g), ds = hr_spinor_bytes(g, HR_BOTH);
    if (cs == 0) return 0;
    return 2 * (2 * up256h(cs) + 2 * up256h(ds)) + up256h(ds / 2);
}

// ops == nullptr: every item applies `op`; else item i applies ops[i] (hr_apply_host_ops: one pipeline across operators)
static int host_pipeline(const hr_geom* g, int op, const int* ops, double m0, const void* u_dev, const void* clover_fwd, const void* clover_inv,
                         int nrhs, const void* const* in_canon_host, void* const* out_canon_host, void* workspace, void* stream) {
    const size_t cs = hr_canonical_spinor_bytes(g), ds = hr_spinor_bytes(g, HR_BOTH), half = ds / 2;
    if (cs == 0) { set_error("hr_apply_host_batch: invalid geometry"); return HR_EINVAL; }
    for (int i = 0; i < (ops ? nrhs : 1); ++i) {
        const int o = ops ? ops[i] : op;
        if (o < HR_EO_HOP_OE || o > HR_HOST_DIRAC) { set_error("hr_apply_host_batch: unknown op %d", o); return HR_EINVAL; }
        if (o == HR_HOST_DIRAC && clover_inv && !ops) { set_error("hr_apply_host_batch: the full operator takes clover_fwd only"); return HR_EINVAL; }
    }
    if (nrhs < 0 || (nrhs > 0 && (!in_canon_host || !out_canon_host))) { set_error("hr_apply_host_batch: nrhs < 0 or NULL pointer arrays"); return HR_EINVAL; }
    if (!u_dev || !workspace || ((uintptr_t)workspace & 15)) { set_error("hr_apply_host_batch: u_dev / workspace NULL or misaligned"); return HR_EINVAL; }
    for (int i = 0; i < nrhs; ++i)
        if (!in_canon_host[i] || !out_canon_host[i]) { set_error("hr_apply_host_batch: host pointer %d is NULL", i); return HR_EINVAL; }
    HostPipe* q = nullptr;
    HR_TRY(pipe_for_current_device(&q));
    cudaStream_t st = (cudaStream_t)stream;
    char* w = (char*)workspace;
    char *c_in[2], *c_out[2], *d_in[2], *d_out[2];
    for (int b = 0; b < 2; ++b) {
        c_in[b] = w; w += up256h(cs);
        c_out[b] = w; w += up256h(cs);
        d_in[b] = w; w += up256h(ds);
        d_out[b] = w; w += up256h(ds);
    }
    char* d_tmp = w;
    // the copy streams start after whatever the caller queued before (it may still be using the workspace)
    HR_CUDA(cudaEventRecord(q->start, st));
    HR_CUDA(cudaStreamWaitEvent(q->s_in, q->start, 0));
    HR_CUDA(cudaStreamWaitEvent(q->s_out, q->start, 0));
    for (int i = 0; i < nrhs; ++i) {
        const int b = i & 1;
        if (ops) op = ops[i];
        // stage 1 (copy-in stream): host -> canonical staging buffer
        if (i >= 2) HR_CUDA(cudaStreamWaitEvent(q->s_in, q->packed[b], 0));      // the pack of spinor i-2 has consumed it
        HR_CUDA(cudaMemcpyAsync(c_in[b], in_canon_host[i], cs, cudaMemcpyHostToDevice, q->s_in));
        HR_CUDA(cudaEventRecord(q->in[b], q->s_in));
        // stage 2 (caller's stream): pack, operator, unpack
        HR_CUDA(cudaStreamWaitEvent(st, q->in[b], 0));
        HR_TRY(hr_pack_spinor(g, c_in[b], d_in[b], stream));
        HR_CUDA(cudaEventRecord(q->packed[b], st));
        if (op == HR_HOST_DIRAC) {
            if (clover_fwd) HR_TRY(hr_dirac_clover_apply(g, u_dev, clover_fwd, d_in[b], d_out[b], stream));   // (clover_inv, if any, belongs to the Dhat items)
            else HR_TRY(hr_dirac_apply(g, m0, u_dev, d_in[b], d_out[b], stream));
        } else {
            HR_CUDA(cudaMemsetAsync(d_out[b], 0, ds, st));                        // the untouched parity comes back as zeros
            const int in_par = (op == HR_EO_HOP_EO) ? HR_ODD : HR_EVEN;
            const int out_par = (op == HR_EO_HOP_OE) ? HR_ODD : HR_EVEN;
            HR_TRY(hr_dirac_eo_apply(g, op, m0, u_dev, clover_fwd, clover_inv, d_in[b] + in_par * half, d_out[b] + out_par * half, d_tmp, stream));
        }
        if (i >= 2) HR_CUDA(cudaStreamWaitEvent(st, q->done[b], 0));              // result i-2 has left the staging buffer
        HR_TRY(hr_unpack_spinor(g, d_out[b], c_out[b], stream));
        HR_CUDA(cudaEventRecord(q->out[b], st));
        // stage 3 (copy-out stream): canonical staging buffer -> host
        HR_CUDA(cudaStreamWaitEvent(q->s_out, q->out[b], 0));
        HR_CUDA(cudaMemcpyAsync(out_canon_host[i], c_out[b], cs, cudaMemcpyDeviceToHost, q->s_out));
        HR_CUDA(cudaEventRecord(q->done[b], q->s_out));
    }
    HR_CUDA(cudaStreamSynchronize(q->s_in));
    HR_CUDA(cudaStreamSynchronize(st));
    HR_CUDA(cudaStreamSynchronize(q->s_out));
    return HR_OK;
}

int hr_apply_host_batch(const hr_geom* g, int op, double m0, const void* u_dev, const void* clover_fwd, const void* clover_inv,
                        int nrhs, const void* const* in_canon_host, void* const* out_canon_host, void* workspace, void* stream) {
    return host_pipeline(g, op, nullptr, m0, u_dev, clover_fwd, clover_inv, nrhs, in_canon_host, out_canon_host, workspace, stream);
}

int hr_apply_host_ops(const hr_geom* g, const int* ops, double m0, const void* u_dev, const void* clover_fwd, const void* clover_inv,
                      int nitems, const void* const* in_canon_host, void* const* out_canon_host, void* workspace, void* stream) {
    if (nitems > 0 && !ops) { set_error("hr_apply_host_ops: ops is NULL"); return HR_EINVAL; }
    return host_pipeline(g, HR_HOST_DIRAC, ops, m0, u_dev, clover_fwd, clover_inv, nitems, in_canon_host, out_canon_host, workspace, stream);
}

}  // extern "C"
