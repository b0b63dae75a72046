// slots.cuh -- the host side of both minimizers: `poll_every` identical slots (evaluation + the
// minimizer's three kernels) are captured ONCE into a CUDA graph and replayed until the device sets
// ctrl->done; between replays the host reads the small control block.  No host decision per iteration
// (BASELINE.json north_star item 4), and at the small configurations, where a slot is ten launches of a
// few microseconds each, no per-launch host cost either.
// Capture needs a capturable stream: the slots run on a stream of the handle's own, ordered after the
// caller's stream by an event on entry and before it by an event on exit (the caller's stream may be the
// legacy default stream, which cannot be captured).
#pragma once
#include "shd_internal.h"

// after_poll(): host hook run after every poll (control block already in h_ctrl, stream idle): fetches the trace ring,
// calls the caller's callback; returns true to stop replaying.
template <class EnqueueSlot, class AfterPoll>
cudaError_t shd_run_slots(shd_ctx* h, int poll_every, EnqueueSlot enqueue_slot, void* h_ctrl, const void* d_ctrl,
                          size_t ctrl_bytes, const int* h_done, AfterPoll after_poll)
{
    cudaError_t e;
    if (!h->gstream) {
        if ((e = cudaStreamCreateWithFlags(&h->gstream, cudaStreamNonBlocking)) != cudaSuccess) return e;
        if ((e = cudaEventCreateWithFlags(&h->gevent, cudaEventDisableTiming)) != cudaSuccess) return e;
    }
    cudaStream_t user = h->stream, gs = h->gstream;
    if ((e = cudaEventRecord(h->gevent, user)) != cudaSuccess) return e;
    if ((e = cudaStreamWaitEvent(gs, h->gevent, 0)) != cudaSuccess) return e;
    h->stream = gs;
    cudaGraph_t graph = nullptr;
    cudaGraphExec_t exec = nullptr;
    e = cudaStreamBeginCapture(gs, cudaStreamCaptureModeThreadLocal);
    if (e == cudaSuccess) {
        cudaError_t le = cudaSuccess;
        for (int k = 0; k < poll_every && le == cudaSuccess; k++) le = enqueue_slot();
        e = cudaStreamEndCapture(gs, &graph);
        if (le != cudaSuccess) e = le;
    }
    if (e == cudaSuccess) e = cudaGraphInstantiate(&exec, graph, 0);
    while (e == cudaSuccess) {
        if ((e = cudaGraphLaunch(exec, gs)) != cudaSuccess) break;
        if ((e = cudaMemcpyAsync(h_ctrl, d_ctrl, ctrl_bytes, cudaMemcpyDeviceToHost, gs)) != cudaSuccess) break;
        if ((e = cudaStreamSynchronize(gs)) != cudaSuccess) break;
        const bool stop = after_poll();
        if (*h_done || stop) break;
    }
    if (exec) cudaGraphExecDestroy(exec);
    if (graph) cudaGraphDestroy(graph);
    h->stream = user;
    if (e == cudaSuccess) e = cudaEventRecord(h->gevent, gs);
    if (e == cudaSuccess) e = cudaStreamWaitEvent(user, h->gevent, 0);
    return e;
}
