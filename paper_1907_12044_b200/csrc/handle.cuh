// handle.cuh -- the opaque tdvp_handle: stream, options, scratch arena, resident chain state.
#pragma once
#include <vector>

#include "common.cuh"

struct StepGraph {                 // a captured TDVP step (CUDA graph), keyed by dt (and one integer: CMF sub-steps)
  cudaGraphExec_t exec = nullptr;
  double dt = 0.0;
  int key = 0;
  long long launches = 0;          // kernels inside the graph (for tdvp_launch_count)
};

struct tdvp_handle {
  cudaStream_t stream = nullptr;
  tdvp_options opt;
  std::string err;
  bool owns_zgemm_ctx = false;     // holds a reference on its stream's GEMM scheduling context
  int *status_dev = nullptr;       // DEVICE: sticky TDVP_STATUS_* bits set by kernels, read by blocking calls
  Arena arena;                     // scratch for the current call (reset per call)
  cudaStream_t copy_stream = nullptr;   // host-entry calls: second H2D queue (created on first use)
  cudaEvent_t ev_first = nullptr, ev_w = nullptr, ev_r = nullptr, ev_l[4] = {nullptr, nullptr, nullptr, nullptr};

  // ---- resident chain state (n == 0 for a context-only handle) ----
  int n = 0;
  std::vector<int> d;              // physical dims [n]
  std::vector<int> Dw;             // MPO bonds [n+1]
  std::vector<int> M;              // MPS bonds [n+1]
  std::vector<c128 *> W;           // dense MPO tensors (DEVICE)
  std::vector<WSparse> Wsp;        // their CSR forms (DEVICE)
  std::vector<void *> Wsp_mem;
  std::vector<c128 *> A;           // MPS tensors (DEVICE)
  std::vector<c128 *> Lenv;        // Lenv[i]: sites < i contracted, [M[i], Dw[i], M[i]]
  std::vector<c128 *> Renv;        // Renv[i]: sites > i contracted, [M[i+1], Dw[i+1], M[i+1]]
  int centre = 0;                  // gauge centre; sites < centre left-canonical, > centre right-canonical
  c128 *tmpA = nullptr;            // scratch site tensors (largest site)
  c128 *tmpB = nullptr;
  c128 *bondD = nullptr;           // bond matrix D and its evolved copy
  c128 *bondD2 = nullptr;
  void *step_ws = nullptr;         // persistent workspace for the step drivers
  size_t step_ws_bytes = 0;
  // TDVP-MU state (allocated on first use)
  std::vector<c128 *> mu_k[7];     // Dormand-Prince stage derivatives
  std::vector<c128 *> mu_y;        // stage states
  double *mu_err_dev = nullptr;
  bool mu_fsal = false;            // mu_k[6] holds the right-hand side at the CURRENT state (first-same-as-last)
  void *mu_scratch = nullptr;      // U, Lambda, V^dagger, centre forms ... of one derivative evaluation
  std::vector<void *> cmf_mem;     // CMF mean fields per bond b: [3b] U, [3b+1] U Lambda, [3b+2] Lambda (first use)
  std::vector<cudaStream_t> cmf_streams;   // side queues of the CMF local propagation, each with scratch
  std::vector<cudaEvent_t> cmf_join, cmf_rel;   // queue q has finished; mean fields of site j are ready
  std::vector<void *> cmf_ws, cmf_scratch;
  cudaEvent_t cmf_fork = nullptr, cmf_hi_done = nullptr;
  cudaStream_t cmf_hi = nullptr;   // highest-priority queue of the CMF mean-field (bond unfolding) chain
  cudaStream_t cmf_env = nullptr;  // queue of what hangs off that chain without being on it: Vh of a bond and the R block built from it
  void *cmf_env_ws = nullptr, *cmf_svd_ws[2] = {nullptr, nullptr};   // its workspace; unfolding workspaces of even / odd bonds
  std::vector<cudaEvent_t> cmf_fac;   // bond i: U, Lambda are ready (the first half of its unfolding is done)
  StepGraph ps_graph, mu_graph, ps2_graph, cmf_graph;
  void *ps2_ws = nullptr;          // two-site TDVP-PS workspace (allocated by the first tdvp_step_ps2)
  size_t ps2_ws_bytes = 0;
};

int set_err(tdvp_handle *h, int code, const std::string &msg);
int check_cuda(tdvp_handle *h, cudaError_t e, const char *what);
// Blocks until the handle's stream is idle, then reports (and clears) what kernels left in status_dev:
// TDVP_ESTATE if a bond SVD did not converge.  Every blocking public call ends here.
int finish_blocking(tdvp_handle *h, const char *what);
tdvp_handle *default_handle();

// Capture `enqueue` into a graph (once per dt and key) and launch it; falls back to direct enqueue when graphs are
// disabled.  Side queues that `enqueue` forks from h->stream by an event and joins again before it returns (the CMF
// local propagation) become parallel branches of the graph.  `enqueue` returns void or a TDVP_E* code.
template <class F>
static inline int run_step(tdvp_handle *h, StepGraph &sg, double dt, F enqueue, const char *what, int key = 0) {
  // (a replayed graph carries no phase brackets: while the phase profiler is on, steps are enqueued directly)
  if ((h->opt.flags & TDVP_FLAG_NO_GRAPH) || g_prof_on.load(std::memory_order_relaxed)) {
    enqueue();
    return check_cuda(h, cudaGetLastError(), what);
  }
  if (!sg.exec || sg.dt != dt || sg.key != key) {
    if (sg.exec) { cudaGraphExecDestroy(sg.exec); sg.exec = nullptr; }
    cudaStream_t cap = h->stream;
    cudaStream_t own = nullptr;
    if (cap == nullptr || cap == cudaStreamLegacy || cap == cudaStreamPerThread) {
      // the legacy default stream cannot be captured: record on a private stream, replay on h->stream
      if (int rc = check_cuda(h, cudaStreamCreateWithFlags(&own, cudaStreamNonBlocking), "stream")) return rc;
      cap = own;
      zgemm_alias_stream(own, h->stream);
    }
    cudaStream_t saved = h->stream;
    h->stream = cap;
    long long tally = 0;
    cudaError_t e = cudaStreamBeginCapture(cap, cudaStreamCaptureModeThreadLocal);
    cudaGraph_t graph = nullptr;
    if (e == cudaSuccess) {
      g_capture_tally = &tally;
      enqueue();
      g_capture_tally = nullptr;
      e = cudaStreamEndCapture(cap, &graph);
    }
    h->stream = saved;
    if (e == cudaSuccess) e = cudaGraphInstantiate(&sg.exec, graph, 0);
    if (graph) cudaGraphDestroy(graph);
    if (own) { zgemm_forget_stream(own); cudaStreamDestroy(own); }
    if (e != cudaSuccess) { sg.exec = nullptr; cudaGetLastError(); return check_cuda(h, e, what); }
    sg.dt = dt; sg.key = key; sg.launches = tally;
  }
  if (int rc = check_cuda(h, cudaGraphLaunch(sg.exec, h->stream), what)) return rc;
  g_launch_count.fetch_add(sg.launches);
  return TDVP_OK;
}

