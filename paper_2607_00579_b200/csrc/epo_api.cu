// Host side of the C ABI declared in include/epo.h: argument validation, host/device pointer
// marshalling, device-memory ownership and launch sequencing.  No arithmetic of the method lives here.
#include <algorithm>
#include <chrono>
#include <cmath>
#include <cstdlib>
#include <cstdarg>
#include <cstring>
#include <new>

#include <nvtx3/nvToolsExt.h>

#include "epo_internal.h"

epo_status epo_fail(epo_ctx* ctx, epo_status st, const char* fmt, ...) {
  if (ctx) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(ctx->err, sizeof(ctx->err), fmt, ap);
    va_end(ap);
  }
  return st;
}

namespace {

// NVTX range around a phase of the public API: shows up as "epo: <call>" on the timeline of a
// profiler that injects NVTX (Nsight Systems / Compute); without one nvtxRangePush is a null function-pointer check.
struct NvtxRange {
  explicit NvtxRange(const char* name) { nvtxRangePushA(name); }
  ~NvtxRange() { nvtxRangePop(); }
  NvtxRange(const NvtxRange&) = delete;
  NvtxRange& operator=(const NvtxRange&) = delete;
};

bool is_device_ptr(const void* p) {
  cudaPointerAttributes a;
  cudaError_t e = cudaPointerGetAttributes(&a, p);
  if (e != cudaSuccess) { cudaGetLastError(); return false; }
  return a.type == cudaMemoryTypeDevice || a.type == cudaMemoryTypeManaged;
}

// EPO_TRACE=1 in the environment: print the wall-clock duration of each phase of a call to stderr (each mark
// drains the stream first, so the phases do not overlap while tracing).  Off: no synchronisation, no output.
struct PhaseTrace {
  cudaStream_t st; const char* what; bool on; std::chrono::steady_clock::time_point t0;
  PhaseTrace(cudaStream_t s, const char* w) : st(s), what(w) {
    const char* v = std::getenv("EPO_TRACE");
    on = v && v[0] && v[0] != '0';
    if (on) { cudaStreamSynchronize(st); t0 = std::chrono::steady_clock::now(); }
  }
  void mark(const char* phase) {
    if (!on) return;
    cudaStreamSynchronize(st);
    auto t1 = std::chrono::steady_clock::now();
    fprintf(stderr, "[epo trace] %s: %-18s %8.3f ms\n", what, phase, std::chrono::duration<double, std::milli>(t1 - t0).count());
    t0 = t1;
  }
};

// copy caller memory (host or device) into library device memory on the context's stream
cudaError_t copy_in(void* dst, const void* src, size_t bytes, cudaStream_t st) {
  return cudaMemcpyAsync(dst, src, bytes, is_device_ptr(src) ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice, st);
}
// copy library device memory to caller memory; *synced is set when the destination is host memory
cudaError_t copy_out(void* dst, const void* src, size_t bytes, cudaStream_t st, bool* need_sync) {
  bool dev = is_device_ptr(dst);
  if (!dev) *need_sync = true;
  return cudaMemcpyAsync(dst, src, bytes, dev ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost, st);
}

void free_views(epo_ctx* c) {
  epo_dfree(c, c->d_edge_off); epo_dfree(c, c->d_edges); epo_dfree(c, c->d_depth);
  c->d_depth = nullptr;
  epo_free_atlas(&c->atlas);
  epo_free_packed(c, &c->packed);
  epo_joint_free(c);
  c->d_edge_off = nullptr; c->d_edges = nullptr;
  c->have_views = false;
}
void destroy_step_graph(epo_ctx* c);
void free_pairs(epo_ctx* c) {
  destroy_step_graph(c);
  epo_dfree(c, c->d_pairs); epo_dfree(c, c->d_perm); epo_dfree(c, c->d_tgt_off); epo_dfree(c, c->d_src_off); epo_dfree(c, c->d_src_inc);
  epo_dfree(c, c->d_work); epo_dfree(c, c->d_work_off); epo_dfree(c, c->d_part); epo_dfree(c, c->d_pair_loss); epo_dfree(c, c->d_pair_valid); epo_dfree(c, c->d_out_f);
  epo_dfree(c, c->d_dz); c->d_dz = nullptr;
  epo_dfree(c, c->d_out_i); epo_dfree(c, c->d_sel_flag); epo_dfree(c, c->d_sel_work); epo_dfree(c, c->d_sel_info); epo_dfree(c, c->d_sel_scratch);
  c->d_sel_scratch = nullptr; c->d_sel_flag = nullptr; c->d_sel_work = nullptr; c->d_sel_info = nullptr; c->subsample = false; c->sel_grid = 0;
  c->d_pairs = nullptr; c->d_perm = nullptr; c->d_tgt_off = nullptr; c->d_src_off = nullptr; c->d_src_inc = nullptr;
  c->d_work = nullptr; c->d_work_off = nullptr; c->d_part = nullptr; c->d_pair_loss = nullptr; c->d_pair_valid = nullptr; c->d_out_f = nullptr;
  c->d_out_i = nullptr;
  c->have_pairs = false; c->P = 0; c->n_work = 0;
}

// Samples per work item (= per CTA) of the fused kernel, a multiple of kLgPass, chosen per problem by simulating the
// launch.  EPO_LG_PASSES in the environment overrides the choice (tuning).
int choose_chunk(const epo_ctx* c, const std::vector<int32_t>& pairs, int64_t P) {
  int sms = 148;
  cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, c->cfg.device);
  const int64_t slots = (int64_t)sms * EPO_LG_MINBLOCKS;
  // passes of every pair; for the simulation below in the order the CTAs are dispatched (canonical: by target, then source)
  std::vector<std::pair<int64_t, int32_t>> order((size_t)P);
  int64_t total_passes = 0;
  for (int64_t k = 0; k < P; ++k) {
    const int32_t s = pairs[2 * k], t = pairs[2 * k + 1];
    order[(size_t)k] = {((int64_t)t << 32) | (uint32_t)s, (c->h_edge_off[s + 1] - c->h_edge_off[s] + kLgPass - 1) / kLgPass};
    total_passes += order[(size_t)k].second;
  }
  // The launch as the block scheduler runs it: items in list order, each to the slot that frees first; an item of p
  // passes holds its slot for t_f + p t_p (measured on B200: 2.1 us of drain, prologue and pipeline refill, 0.62 us per
  // pass at full residency).  Short items pay t_f too often, long ones quantise the last wave: take the
  // item length with the shortest simulated launch.  Time in units of t_p / 5 (t_f = 17 units), so that the slots' free
  // times are integers and a calendar of counters replaces a priority queue; with eight or more full waves at the
  // longest item the quantisation is immaterial and the longest item wins without a simulation.
  int best = kLgMaxOuter;
  if (total_passes < slots * kLgMaxOuter * 8) {
    std::sort(order.begin(), order.end());
    constexpr int kTf = 17, kTp = 5;
    int64_t best_t = INT64_MAX;
    std::vector<int32_t> cal;
    for (int maxp = 4; maxp <= kLgMaxOuter; maxp += (maxp < 24 ? 1 : 4)) {
      const int64_t horizon = (total_passes * kTp + (total_passes / maxp + P) * kTf) / slots + 2 * (kTf + kLgMaxOuter * kTp) + 2;
      cal.assign((size_t)horizon + kTf + kLgMaxOuter * kTp + 2, 0);
      cal[0] = (int32_t)slots;
      int64_t cur = 0, end = 0;
      auto run_item = [&](int passes) {
        while (cal[(size_t)cur] == 0) ++cur;
        --cal[(size_t)cur];
        const int64_t t = cur + kTf + (int64_t)passes * kTp;
        if ((size_t)t >= cal.size()) cal.resize((size_t)t + 64, 0);
        ++cal[(size_t)t];
        if (t > end) end = t;
      };
      for (const auto& o : order) {
        int left = o.second;
        for (; left > maxp; left -= maxp) run_item(maxp);
        if (left > 0) run_item(left);
      }
      if (end * 200 < best_t * 199) { best_t = end; best = maxp; }     // near-ties: the shorter item
    }
  }
  if (const char* v = std::getenv("EPO_LG_PASSES")) { int k = std::atoi(v); if (k >= 1 && k <= kLgMaxOuter) best = k; }
  return best * kLgPass;
}

void destroy_step_graph(epo_ctx* c) {
  if (c->step_exec) cudaGraphExecDestroy(c->step_exec);
  if (c->step_graph) cudaGraphDestroy(c->step_graph);
  c->step_exec = nullptr; c->step_graph = nullptr; c->step_begin_node = nullptr; c->step_cond = 0;
}

// One iteration as the loop enqueues it: [select pairs] -> fused -> finish -> [joint points], every kernel self-gated
// by DevState.halt, chained by programmatic dependent launch.
epo_status enqueue_iteration(epo_ctx* c, cudaGraphConditionalHandle cond) {
  const bool joint = c->cfg.joint_phase != 0;
  if (c->subsample) EPO_TRY(epo_launch_select_pairs(c, -1, true, true));
  EPO_TRY(epo_launch_fused(c, -1.0f, true, c->subsample, joint));
  EPO_TRY(epo_launch_finish(c, true, true, c->subsample, joint, cond));
  // joint phase: AdamW on (alpha, beta) where due and the points again from the new K and Z (gamma was stepped in
  // k_finish); self-gated by DevState.joint_pending
  if (joint) EPO_TRY(epo_launch_joint_points(c, c->subsample));
  return EPO_OK;
}

// The whole epo_step call as one graph: k_begin_step_call (iteration budget, initial condition) -> WHILE(condition)
// { graph_unroll iterations }.  The body is captured from the very launches the host loop would issue, so the
// programmatic-dependent-launch edges between its kernels are kept; k_finish sets the condition, and once it is 0
// nothing more is launched (PAPER.md:436-446 is a host `break`; SURVEY.md section 3 "a CUDA-graph conditional loop").
// On any failure the context falls back to the host loop (use_graph = false).
epo_status build_step_graph(epo_ctx* c) {
  destroy_step_graph(c);
  cudaError_t e = cudaGraphCreate(&c->step_graph, 0);
  if (e == cudaSuccess) e = cudaGraphConditionalHandleCreate(&c->step_cond, c->step_graph, 0, 0);
  EpoBeginArgs ba;
  if (e == cudaSuccess) {
    epo_begin_step_call_args(c, 0, 0, c->step_cond, &ba);
    cudaKernelNodeParams kp = {};
    kp.func = ba.func; kp.gridDim = dim3(1); kp.blockDim = dim3(1); kp.sharedMemBytes = 0; kp.kernelParams = ba.ptrs; kp.extra = nullptr;
    e = cudaGraphAddKernelNode(&c->step_begin_node, c->step_graph, nullptr, 0, &kp);
  }
  cudaGraph_t body = nullptr;
  if (e == cudaSuccess) {
    cudaGraphNodeParams cp = {};
    cp.type = cudaGraphNodeTypeConditional;
    cp.conditional.handle = c->step_cond; cp.conditional.type = cudaGraphCondTypeWhile; cp.conditional.size = 1;
    cudaGraphNode_t cnode = nullptr;
    e = cudaGraphAddNode(&cnode, c->step_graph, &c->step_begin_node, 1, &cp);
    if (e == cudaSuccess) body = cp.conditional.phGraph_out[0];
  }
  epo_status rc = EPO_OK;
  if (e == cudaSuccess) {
    // capture the iterations on a private stream (the caller's may be the legacy default stream, which cannot capture)
    cudaStream_t user = c->stream;
    const int64_t launches = c->launches;
    const bool dirty = c->static_dirty;
    c->static_dirty = false;                         // inside the graph every launch follows the loop's own kernels
    e = cudaStreamBeginCaptureToGraph(c->capture_stream, body, nullptr, nullptr, 0, cudaStreamCaptureModeRelaxed);
    if (e == cudaSuccess) {
      c->stream = c->capture_stream;
      for (int u = 0; u < c->graph_unroll && rc == EPO_OK; ++u) rc = enqueue_iteration(c, c->step_cond);
      c->stream = user;
      cudaGraph_t got = nullptr;
      e = cudaStreamEndCapture(c->capture_stream, &got);
    }
    c->launches = launches; c->static_dirty = dirty;
  }
  if (e == cudaSuccess && rc == EPO_OK) e = cudaGraphInstantiate(&c->step_exec, c->step_graph, 0);
  if (e != cudaSuccess || rc != EPO_OK) {
    cudaGetLastError();
    destroy_step_graph(c);
    c->use_graph = false;
    if (std::getenv("EPO_TRACE")) fprintf(stderr, "[epo trace] loop graph unavailable (%s): host launch loop\n", cudaGetErrorString(e));
  }
  return EPO_OK;
}

epo_status reset_optimiser(epo_ctx* c, bool joint = true) {
  cudaStream_t st = c->stream;
  if (joint) EPO_TRY(epo_joint_reset(c));
  EPO_CUDA(c, cudaMemsetAsync(c->d_m, 0, (size_t)c->N * 6 * sizeof(double), st));
  EPO_CUDA(c, cudaMemsetAsync(c->d_v, 0, (size_t)c->N * 6 * sizeof(double), st));
  EPO_CUDA(c, cudaMemsetAsync(c->d_state, 0, sizeof(DevState), st));
  EPO_CUDA(c, cudaMemsetAsync(c->d_theta, 0, (size_t)c->cfg.max_steps * sizeof(double), st));
  EPO_CUDA(c, cudaMemsetAsync(c->d_loss_trace, 0, (size_t)c->cfg.max_steps * sizeof(double), st));
  return EPO_OK;
}

}  // namespace

extern "C" {

const char* epo_version(void) { return "epo-b200 0.1 (sm_100a)"; }

const char* epo_last_error(const epo_ctx* ctx) { return ctx ? ctx->err : "null context"; }

epo_status epo_config_default(epo_config* cfg) {
  if (!cfg) return EPO_ERR_INVALID_ARG;
  std::memset(cfg, 0, sizeof(*cfg));
  cfg->huber_delta = 1.0f;
  cfg->clamp_start = 10.0f; cfg->clamp_end = 6.0f; cfg->clamp_steps = 1000;
  cfg->lr_max = 3e-3f; cfg->warmup_steps = 25; cfg->max_steps = 2000;
  cfg->beta1 = 0.9f; cfg->beta2 = 0.999f; cfg->adam_eps = 1e-8f;
  cfg->eps1 = 0.5f; cfg->eps2 = 0.1f; cfg->w1 = 25; cfg->w2 = 50;
  cfg->smooth_window = 1; cfg->early_stop = 1; cfg->dtf_format = 0; cfg->e_max = 0;
  cfg->z_min = 1e-6f; cfg->device = 0; cfg->stream = nullptr;
  cfg->pair_budget = 0; cfg->subsample_seed = 0;
  cfg->stop_rule = 0; cfg->w_loss = 100; cfg->eps_loss = 5e-4f;
  cfg->joint_phase = 0; cfg->weight_decay = 0.01f;
  cfg->mem_pool = nullptr;
  return EPO_OK;
}

epo_status epo_create(const epo_config* cfg, epo_ctx** out) {
  if (!cfg || !out) return EPO_ERR_INVALID_ARG;
  *out = nullptr;
  if (cfg->n_views < 2 || cfg->n_views > 65535 || cfg->width < 2 || cfg->height < 2 || cfg->width > 65535 || cfg->height > 65535)
    return EPO_ERR_INVALID_ARG;
  if (!(cfg->huber_delta > 0.f) || cfg->clamp_steps < 1 || cfg->warmup_steps < 0 || cfg->max_steps <= cfg->warmup_steps ||
      cfg->w1 < 1 || cfg->w2 < 1 || (cfg->dtf_format != 0 && cfg->dtf_format != 1) || cfg->e_max < 0 ||
      cfg->pair_budget < 0 || (cfg->joint_phase != 0 && cfg->joint_phase != 1) || !(cfg->weight_decay >= 0.f) ||
      (cfg->stop_rule != 0 && cfg->stop_rule != 1) || cfg->w_loss < 1 || !(cfg->eps_loss >= 0.f) || !(cfg->beta1 >= 0.f && cfg->beta1 < 1.f) || !(cfg->beta2 >= 0.f && cfg->beta2 < 1.f) || !(cfg->z_min >= 0.f))
    return EPO_ERR_INVALID_ARG;
  epo_ctx* c = new (std::nothrow) epo_ctx();
  if (!c) return EPO_ERR_OUT_OF_MEMORY;
  c->cfg = *cfg; c->stream = (cudaStream_t)cfg->stream;
  c->N = cfg->n_views; c->W = cfg->width; c->H = cfg->height;
  c->have_views = c->have_pairs = false; c->P = c->E = c->n_work = c->reproj_per_eval = c->launches = 0; c->lg_chunk = kLgOuter * kLgPass;
  c->err[0] = 0;
  c->pool = nullptr; c->own_pool = false;
  c->atlas = EpoAtlas{nullptr, nullptr, 0, 0, 1};
  c->packed.xyz = nullptr; c->packed.pix = nullptr; c->packed.d_off = nullptr;
  { const char* v = std::getenv("EPO_NO_GRAPH"); c->use_graph = !(v && v[0] && v[0] != '0'); }
  c->graph_unroll = 8;
  if (const char* v = std::getenv("EPO_GRAPH_UNROLL")) { const int k = std::atoi(v); if (k >= 1 && k <= 64) c->graph_unroll = k; }
  c->capture_stream = nullptr; c->step_graph = nullptr; c->step_exec = nullptr; c->step_begin_node = nullptr; c->step_cond = 0;
  { const char* v = std::getenv("EPO_NO_PDL"); c->pdl = !(v && v[0] && v[0] != '0'); }
  { const char* v = std::getenv("EPO_NO_COOP"); c->coop_select = !(v && v[0] && v[0] != '0'); }
  c->static_dirty = true;
  cudaError_t e = cudaSetDevice(cfg->device);
  const size_t N = (size_t)c->N;
  if (e == cudaSuccess) {
    if (cfg->mem_pool) {
      c->pool = (cudaMemPool_t)cfg->mem_pool;       // caller-owned: shared between contexts, never destroyed here
    } else {
      // a private pool that keeps freed blocks until epo_destroy (no process-wide side effect)
      cudaMemPoolProps props = {};
      props.allocType = cudaMemAllocationTypePinned; props.handleTypes = cudaMemHandleTypeNone;
      props.location.type = cudaMemLocationTypeDevice; props.location.id = cfg->device;
      e = cudaMemPoolCreate(&c->pool, &props);
      if (e == cudaSuccess) {
        c->own_pool = true;
        unsigned long long keep = ~0ull;
        e = cudaMemPoolSetAttribute(c->pool, cudaMemPoolAttrReleaseThreshold, &keep);
      }
    }
  }
  if (e == cudaSuccess) {
    e = cudaStreamCreateWithFlags(&c->copy_stream, cudaStreamNonBlocking);
    if (e == cudaSuccess) e = cudaStreamCreateWithFlags(&c->capture_stream, cudaStreamNonBlocking);
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&c->ev_alloc, cudaEventDisableTiming);
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&c->ev_copied, cudaEventDisableTiming);
  }
  if (e == cudaSuccess) e = epo_dmalloc(c, &c->d_K, N * 4 * sizeof(float));
  if (e == cudaSuccess) e = epo_dmalloc(c, &c->d_poses, N * 12 * sizeof(double));
  if (e == cudaSuccess) e = epo_dmalloc(c, &c->d_poses_next, N * 12 * sizeof(double));
  if (e == cudaSuccess) e = epo_dmalloc(c, &c->d_poses_init, N * 12 * sizeof(double));
  if (e == cudaSuccess) e = epo_dmalloc(c, &c->d_grad, N * 6 * sizeof(double));
  if (e == cudaSuccess) e = epo_dmalloc(c, &c->d_loss_part, N * sizeof(double));
  if (e == cudaSuccess) e = epo_dmalloc(c, &c->d_m, N * 6 * sizeof(double));
  if (e == cudaSuccess) e = epo_dmalloc(c, &c->d_v, N * 6 * sizeof(double));
  if (e == cudaSuccess) e = epo_dmalloc(c, &c->d_dR, N * sizeof(double));
  if (e == cudaSuccess) e = epo_dmalloc(c, &c->d_dt, N * sizeof(double));
  if (e == cudaSuccess) e = epo_dmalloc(c, &c->d_state, sizeof(DevState));
  if (e == cudaSuccess) e = epo_dmalloc(c, &c->d_sched, (size_t)cfg->max_steps * 4 * sizeof(double));
  if (e == cudaSuccess) e = epo_dmalloc(c, &c->d_theta, (size_t)cfg->max_steps * sizeof(double));
  if (e == cudaSuccess) e = epo_dmalloc(c, &c->d_loss_trace, (size_t)cfg->max_steps * sizeof(double));
  if (e != cudaSuccess) {
    epo_status st = (e == cudaErrorMemoryAllocation) ? EPO_ERR_OUT_OF_MEMORY : EPO_ERR_CUDA;
    cudaGetLastError();
    epo_destroy(c);
    return st;
  }
  if (epo_launch_fill_schedule(c) != EPO_OK) { epo_destroy(c); return EPO_ERR_CUDA; }
  *out = c;
  return EPO_OK;
}

void epo_destroy(epo_ctx* c) {
  if (!c) return;
  cudaSetDevice(c->cfg.device);
  cudaStreamSynchronize(c->stream);
  free_pairs(c); free_views(c);
  epo_dfree(c, c->d_K); epo_dfree(c, c->d_poses); epo_dfree(c, c->d_poses_next); epo_dfree(c, c->d_poses_init); epo_dfree(c, c->d_grad); epo_dfree(c, c->d_loss_part);
  epo_dfree(c, c->d_m); epo_dfree(c, c->d_v); epo_dfree(c, c->d_dR); epo_dfree(c, c->d_dt); epo_dfree(c, c->d_state);
  epo_dfree(c, c->d_sched); epo_dfree(c, c->d_theta); epo_dfree(c, c->d_loss_trace);
  cudaStreamSynchronize(c->stream);                 // the frees are stream-ordered: done before the context goes
  if (c->own_pool && c->pool) cudaMemPoolDestroy(c->pool);
  if (c->copy_stream) cudaStreamDestroy(c->copy_stream);
  if (c->capture_stream) cudaStreamDestroy(c->capture_stream);
  if (c->ev_alloc) cudaEventDestroy(c->ev_alloc);
  if (c->ev_copied) cudaEventDestroy(c->ev_copied);
  cudaGetLastError();
  delete c;
}

epo_status epo_set_views(epo_ctx* c, const float* K, const float* poses, const float* depth, const uint8_t* edges) {
  if (!c) return EPO_ERR_INVALID_ARG;
  NvtxRange nvtx_("epo: epo_set_views");
  if (!K || !poses || !depth || !edges) return epo_fail(c, EPO_ERR_INVALID_ARG, "epo_set_views: NULL argument");
  EPO_CUDA(c, cudaSetDevice(c->cfg.device));
  cudaStream_t st = c->stream;
  const size_t N = (size_t)c->N, px = (size_t)c->W * c->H;
  // validate intrinsics and poses on the host (small arrays)
  std::vector<float> hK(N * 4), hP(N * 12);
  EPO_CUDA(c, cudaMemcpyAsync(hK.data(), K, N * 4 * sizeof(float), cudaMemcpyDefault, st));
  EPO_CUDA(c, cudaMemcpyAsync(hP.data(), poses, N * 12 * sizeof(float), cudaMemcpyDefault, st));
  EPO_CUDA(c, cudaStreamSynchronize(st));
  for (size_t i = 0; i < N; ++i) {
    if (!(std::isfinite(hK[4 * i]) && hK[4 * i] > 0.f && std::isfinite(hK[4 * i + 1]) && hK[4 * i + 1] > 0.f &&
          std::isfinite(hK[4 * i + 2]) && std::isfinite(hK[4 * i + 3])))
      return epo_fail(c, EPO_ERR_INVALID_ARG, "epo_set_views: view %zu has non-finite or non-positive intrinsics", i);
    for (int k = 0; k < 12; ++k)
      if (!std::isfinite(hP[12 * i + k]))
        return epo_fail(c, EPO_ERR_INVALID_ARG, "epo_set_views: view %zu has a non-finite pose", i);
  }
  // build everything into temporaries; commit only on success (all-or-nothing)
  PhaseTrace tr(st, "epo_set_views");
  float* d_depth = nullptr; uint8_t* d_e = nullptr; float* d_small = nullptr;
  int32_t* off = nullptr; EdgeRec* rec = nullptr; int64_t E = 0;
  EpoAtlas atlas = {nullptr, nullptr, 0, 0, 1};
  EpoPacked packed = {nullptr, nullptr, nullptr, {}};
  EpoDtfScratch scratch = {nullptr, 0, 0};
  std::vector<int32_t> hoff;
  bool subsampled = false;
  epo_status rc = EPO_OK;
  cudaError_t e = epo_dmalloc(c, &d_depth, N * px * sizeof(float));
  if (e == cudaSuccess) e = epo_dmalloc(c, &d_e, N * px);
  if (e == cudaSuccess) e = epo_dmalloc(c, &d_small, N * 16 * sizeof(float));   // [K 4N | poses 12N] staging
  tr.mark("alloc inputs");
  // the depth maps travel on the copy stream while the edge maps arrive and the distance transform runs here
  bool depth_in_flight = false;
  if (e == cudaSuccess) e = cudaEventRecord(c->ev_alloc, st);
  if (e == cudaSuccess) e = copy_in(d_e, edges, N * px, st);      // issued first: the link serves it first
  if (e == cudaSuccess) e = cudaStreamWaitEvent(c->copy_stream, c->ev_alloc, 0);
  if (e == cudaSuccess) { e = copy_in(d_depth, depth, N * px * sizeof(float), c->copy_stream); depth_in_flight = true; }
  if (e == cudaSuccess) e = cudaEventRecord(c->ev_copied, c->copy_stream);
  if (e == cudaSuccess) e = cudaMemcpyAsync(d_small, hK.data(), N * 4 * sizeof(float), cudaMemcpyHostToDevice, st);
  if (e == cudaSuccess) e = cudaMemcpyAsync(d_small + N * 4, hP.data(), N * 12 * sizeof(float), cudaMemcpyHostToDevice, st);
  if (e != cudaSuccess)
    rc = epo_fail(c, e == cudaErrorMemoryAllocation ? EPO_ERR_OUT_OF_MEMORY : EPO_ERR_CUDA, "epo_set_views: %s",
                  cudaGetErrorString(e));
  tr.mark("copy edges");
  if (rc == EPO_OK) rc = epo_build_dtf_atlas(c, d_e, &atlas, &scratch);
  tr.mark("distance fields");
  if (depth_in_flight) {
    // whatever happened above, this stream goes on (or frees d_depth) only after the copy has landed
    e = cudaStreamWaitEvent(st, c->ev_copied, 0);
    if (e != cudaSuccess) { cudaStreamSynchronize(c->copy_stream); if (rc == EPO_OK) rc = epo_fail(c, EPO_ERR_CUDA, "epo_set_views: %s", cudaGetErrorString(e)); }
  }
  tr.mark("copy depth");
  if (rc == EPO_OK) rc = epo_build_edge_lists(c, d_e, d_depth, &off, &rec, &E, &hoff, &subsampled);
  tr.mark("edge lists");
  if (rc == EPO_OK) rc = epo_build_points(c, d_small, off, rec, E, hoff, d_e, d_depth, subsampled, &packed);
  if (rc == EPO_OK) {
    // commit the small state on the stream, then drain it once
    e = cudaMemcpyAsync(c->d_K, d_small, N * 4 * sizeof(float), cudaMemcpyDeviceToDevice, st);
    if (e == cudaSuccess) {
      epo_launch_f32_to_f64(st, d_small + N * 4, c->d_poses_init, (int64_t)N * 12);
      c->launches += 1;
      e = cudaMemcpyAsync(c->d_poses, c->d_poses_init, N * 12 * sizeof(double), cudaMemcpyDeviceToDevice, st);
    }
    if (e == cudaSuccess) e = cudaGetLastError();
    if (e != cudaSuccess) rc = epo_fail(c, EPO_ERR_CUDA, "epo_set_views: %s", cudaGetErrorString(e));
  }
  if (rc == EPO_OK) rc = reset_optimiser(c, false);
  e = cudaStreamSynchronize(st);
  if (rc == EPO_OK && e != cudaSuccess) rc = epo_fail(c, EPO_ERR_CUDA, "epo_set_views: %s", cudaGetErrorString(e));
  tr.mark("points + drain");
  epo_free_dtf_scratch(c, &scratch);
  epo_dfree(c, d_e); epo_dfree(c, d_small);
  if (rc != EPO_OK) {
    epo_dfree(c, d_depth);
    // d_K / d_poses may have been overwritten only if every build step succeeded and the final drain failed
    // (a sticky CUDA error: the context is unusable anyway)
    cudaGetLastError();
    epo_dfree(c, off); epo_dfree(c, rec); epo_free_atlas(&atlas); epo_free_packed(c, &packed);
    return rc;
  }
  free_pairs(c); free_views(c);
  c->d_edge_off = off; c->d_edges = rec; c->E = E; c->h_edge_off = hoff;
  c->atlas = atlas; c->d_depth = d_depth; c->packed = packed;
  c->have_views = true; c->static_dirty = true;
  EPO_TRY(epo_joint_alloc(c));                      // joint loop: variables at the identity, Z0 and K0 kept
  tr.mark("free temporaries");
  return EPO_OK;
}

epo_status epo_set_pairs(epo_ctx* c, const int32_t* pairs, int64_t P) {
  if (!c) return EPO_ERR_INVALID_ARG;
  NvtxRange nvtx_("epo: epo_set_pairs");
  if (!c->have_views) return epo_fail(c, EPO_ERR_BAD_STATE, "epo_set_pairs before epo_set_views");
  if (!pairs || P <= 0 || P > (int64_t)1 << 30) return epo_fail(c, EPO_ERR_INVALID_ARG, "epo_set_pairs: NULL list or bad count");
  EPO_CUDA(c, cudaSetDevice(c->cfg.device));
  cudaStream_t st = c->stream;
  std::vector<int32_t> hp((size_t)P * 2);
  EPO_CUDA(c, cudaMemcpyAsync(hp.data(), pairs, (size_t)P * 2 * sizeof(int32_t), cudaMemcpyDefault, st));
  EPO_CUDA(c, cudaStreamSynchronize(st));
  int64_t reproj = 0;
  for (int64_t k = 0; k < P; ++k) {
    int s = hp[2 * k], t = hp[2 * k + 1];
    if (s < 0 || s >= c->N || t < 0 || t >= c->N || s == t)
      return epo_fail(c, EPO_ERR_INVALID_ARG, "epo_set_pairs: pair %lld = (%d, %d) is invalid", (long long)k, s, t);
    reproj += c->h_edge_off[s + 1] - c->h_edge_off[s];
  }
  int32_t* d_user = nullptr;
  EPO_CUDA(c, epo_dmalloc(c, &d_user, (size_t)P * 2 * sizeof(int32_t)));
  cudaError_t e = cudaMemcpyAsync(d_user, hp.data(), (size_t)P * 2 * sizeof(int32_t), cudaMemcpyHostToDevice, st);
  int2* canon = nullptr; int4* work = nullptr; int32_t *perm = nullptr, *toff = nullptr, *soff = nullptr, *sinc = nullptr, *woff = nullptr;
  int64_t n_work = 0;
  const int chunk = choose_chunk(c, hp, P);
  epo_status rc = (e == cudaSuccess) ? epo_build_pairs(c, d_user, P, &canon, &perm, &toff, &soff, &sinc, &work, &woff, &n_work, chunk)
                                     : epo_fail(c, EPO_ERR_CUDA, "epo_set_pairs: %s", cudaGetErrorString(e));
  epo_dfree(c, d_user);
  double* acc = nullptr; float* pl = nullptr; int32_t* pv = nullptr; float* of = nullptr; int32_t* oi = nullptr; float2* dz = nullptr;
  uint8_t* sflag = nullptr; int32_t* swork = nullptr; int32_t* sinfo = nullptr; int32_t* sscr = nullptr;
  if (rc == EPO_OK && c->cfg.pair_budget > 0 && P > c->cfg.pair_budget) {
    // k_select_pairs meets at grid barriers: all its CTAs (4096 pairs each) must be resident at once, one per SM
    int sms = 148;
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, c->cfg.device);
    const int64_t max_pairs = std::min<int64_t>(epo_select_max_pairs(), (int64_t)sms * 4096);
    if (P > max_pairs) rc = epo_fail(c, EPO_ERR_UNSUPPORTED, "pair sub-sampling supports at most %lld pairs", (long long)max_pairs);
  }
  if (rc == EPO_OK) {
    e = epo_dmalloc(c, &sscr, (size_t)kSelScrInts * sizeof(int32_t));
    if (e == cudaSuccess) e = cudaMemsetAsync(sscr, 0, (size_t)kSelScrInts * sizeof(int32_t), st);
    if (e != cudaSuccess) rc = epo_fail(c, EPO_ERR_CUDA, "epo_set_pairs: %s", cudaGetErrorString(e));
  }
  if (rc == EPO_OK) {
    e = epo_dmalloc(c, &sflag, (size_t)P);
    if (e == cudaSuccess) e = epo_dmalloc(c, &swork, (size_t)(n_work > 0 ? n_work : 1) * sizeof(int32_t));
    if (e == cudaSuccess) e = epo_dmalloc(c, &sinfo, 2 * sizeof(int32_t));
    if (e == cudaSuccess) e = cudaMemsetAsync(sinfo, 0, 2 * sizeof(int32_t), st);
    if (e != cudaSuccess)
      rc = epo_fail(c, e == cudaErrorMemoryAllocation ? EPO_ERR_OUT_OF_MEMORY : EPO_ERR_CUDA, "epo_set_pairs: %s",
                    cudaGetErrorString(e));
  }
  if (rc == EPO_OK) {
    // output staging: [loss | grad 6N | pair_loss P | loss trace | theta trace]
    size_t nf = 1 + (size_t)c->N * 6 + (size_t)P + (size_t)c->cfg.max_steps * 2;
    // partial records at the joint phase's stride (epo_loss_grad_joint works in every context)
    e = epo_dmalloc(c, &acc, (size_t)(n_work > 0 ? n_work : 1) * kAccStrideJoint * sizeof(double));
    if (e == cudaSuccess && c->cfg.joint_phase) e = epo_dmalloc(c, &dz, (size_t)(n_work > 0 ? n_work : 1) * (size_t)(chunk / 2) * sizeof(float2));
    if (e == cudaSuccess) e = epo_dmalloc(c, &pl, (size_t)P * sizeof(float));
    if (e == cudaSuccess) e = epo_dmalloc(c, &pv, (size_t)P * sizeof(int32_t));
    if (e == cudaSuccess) e = epo_dmalloc(c, &of, nf * sizeof(float));
    if (e == cudaSuccess) e = epo_dmalloc(c, &oi, (size_t)P * sizeof(int32_t));
    if (e != cudaSuccess)
      rc = epo_fail(c, e == cudaErrorMemoryAllocation ? EPO_ERR_OUT_OF_MEMORY : EPO_ERR_CUDA, "epo_set_pairs: %s",
                    cudaGetErrorString(e));
  }
  if (rc != EPO_OK) {
    cudaGetLastError();
    epo_dfree(c, canon); epo_dfree(c, work); epo_dfree(c, perm); epo_dfree(c, toff); epo_dfree(c, soff); epo_dfree(c, sinc); epo_dfree(c, woff);
    epo_dfree(c, acc); epo_dfree(c, pl); epo_dfree(c, pv); epo_dfree(c, of); epo_dfree(c, oi); epo_dfree(c, dz);
    epo_dfree(c, sflag); epo_dfree(c, swork); epo_dfree(c, sinfo); epo_dfree(c, sscr);
    return rc;
  }
  free_pairs(c);
  c->d_pairs = canon; c->d_perm = perm; c->d_tgt_off = toff; c->d_src_off = soff; c->d_src_inc = sinc; c->d_work = work;
  c->d_work_off = woff; c->n_work = n_work; c->P = P; c->d_part = acc; c->d_pair_loss = pl; c->d_pair_valid = pv; c->d_out_f = of; c->d_out_i = oi;
  c->h_pairs.swap(hp); c->reproj_per_eval = reproj; c->lg_chunk = chunk;
  c->d_sel_flag = sflag; c->d_sel_work = swork; c->d_sel_info = sinfo; c->d_sel_scratch = sscr; c->d_dz = dz;
  // stochastic pair sub-sampling: only when the list is longer than the budget (Alg. 3 l.3-6)
  c->subsample = c->cfg.pair_budget > 0 && P > c->cfg.pair_budget;
  {
    int64_t max_items = 1;   // work items of the longest pair
    for (int64_t k = 0; k < P; ++k) {
      const int64_t n = c->h_edge_off[c->h_pairs[2 * k] + 1] - c->h_edge_off[c->h_pairs[2 * k]];
      const int64_t it = (n + chunk - 1) / chunk;
      if (it > max_items) max_items = it;
    }
    c->sel_grid = (int64_t)c->cfg.pair_budget * max_items;
    if (c->sel_grid > n_work) c->sel_grid = n_work;
    if (c->sel_grid < 1) c->sel_grid = 1;
  }
  c->have_pairs = true; c->static_dirty = true;
  // the optimiser restarts (moments, step counter, phase, traces); the CURRENT poses and joint variables stay, so that
  // a viewgraph re-estimated with epo_build_viewgraph from refined poses can be installed without losing them
  EPO_TRY(reset_optimiser(c, false));
  EPO_TRY(epo_joint_reset_moments(c));
  return EPO_OK;
}

epo_status epo_loss_grad(epo_ctx* c, float lambda, float* loss, float* pair_loss, int32_t* pair_valid, float* grad) {
  if (!c) return EPO_ERR_INVALID_ARG;
  NvtxRange nvtx_("epo: epo_loss_grad");
  if (!c->have_views || !c->have_pairs) return epo_fail(c, EPO_ERR_BAD_STATE, "epo_loss_grad before epo_set_views/epo_set_pairs");
  if (!loss || !(lambda >= 0.f)) return epo_fail(c, EPO_ERR_INVALID_ARG, "epo_loss_grad: NULL loss or negative lambda");
  EPO_CUDA(c, cudaSetDevice(c->cfg.device));
  cudaStream_t st = c->stream;
  EPO_TRY(epo_launch_fused(c, lambda, false, false, false));
  EPO_TRY(epo_launch_finish(c, false, false, false, false, 0));
  bool sync = false;
  // loss: DevState.loss (double) -> float
  epo_launch_f64_to_f32(st, &c->d_state->loss, c->d_out_f, 1);
  EPO_CUDA(c, copy_out(loss, c->d_out_f, sizeof(float), st, &sync));
  if (grad) {
    epo_launch_f64_to_f32(st, c->d_grad, c->d_out_f + 1, (int64_t)c->N * 6);
    EPO_CUDA(c, copy_out(grad, c->d_out_f + 1, (size_t)c->N * 6 * sizeof(float), st, &sync));
    c->launches += 1;
  }
  c->launches += 1;
  if (pair_loss || pair_valid) {
    // user-order outputs: written straight into device destinations, staged in d_out_f / d_out_i for host ones
    float* stage_pl = c->d_out_f + 1 + (size_t)c->N * 6;
    float* opl = pair_loss ? (is_device_ptr(pair_loss) ? pair_loss : stage_pl) : nullptr;
    int32_t* opv = pair_valid ? (is_device_ptr(pair_valid) ? pair_valid : c->d_out_i) : nullptr;
    epo_launch_scatter_pair_outputs(st, c->d_pair_loss, c->d_pair_valid, c->d_perm, opl, opv, c->P);
    c->launches += 1;
    if (opl == stage_pl) EPO_CUDA(c, copy_out(pair_loss, stage_pl, (size_t)c->P * sizeof(float), st, &sync));
    if (opv == c->d_out_i) EPO_CUDA(c, copy_out(pair_valid, c->d_out_i, (size_t)c->P * sizeof(int32_t), st, &sync));
  }
  if (sync) EPO_CUDA(c, cudaStreamSynchronize(st));
  EPO_CUDA(c, cudaGetLastError());
  return EPO_OK;
}

epo_status epo_loss_grad_joint(epo_ctx* c, float lambda, float* loss, float* g_logf, float* g_depth) {
  if (!c) return EPO_ERR_INVALID_ARG;
  NvtxRange nvtx_("epo: epo_loss_grad_joint");
  if (!c->have_views || !c->have_pairs) return epo_fail(c, EPO_ERR_BAD_STATE, "epo_loss_grad_joint before epo_set_views/epo_set_pairs");
  if (!g_logf || !g_depth || !(lambda >= 0.f)) return epo_fail(c, EPO_ERR_INVALID_ARG, "epo_loss_grad_joint: NULL output or negative lambda");
  EPO_CUDA(c, cudaSetDevice(c->cfg.device));
  cudaStream_t st = c->stream;
  const size_t N = (size_t)c->N, px = N * c->W * c->H;
  // one pass of the fused kernel in joint mode (loss, pose gradient, the focal sums and a . t_ts of every sample), the
  // per-camera reduction (valid counts, d L / d ln f), then every edge pixel's pairs summed into the dense map
  float2* dz = c->d_dz; float2* dz_tmp = nullptr; float* d_gf32 = nullptr; float* d_gz = nullptr;
  const bool gz_dev = is_device_ptr(g_depth);
  cudaError_t e = epo_dmalloc(c, &d_gf32, N * sizeof(float));
  if (e == cudaSuccess && !dz) {
    e = epo_dmalloc(c, &dz_tmp, (size_t)(c->n_work > 0 ? c->n_work : 1) * (size_t)(c->lg_chunk / 2) * sizeof(float2));
    dz = dz_tmp;
  }
  if (e == cudaSuccess && !gz_dev) e = epo_dmalloc(c, &d_gz, px * sizeof(float));
  epo_status rc = e == cudaSuccess ? EPO_OK : epo_fail(c, e == cudaErrorMemoryAllocation ? EPO_ERR_OUT_OF_MEMORY : EPO_ERR_CUDA,
                                                        "epo_loss_grad_joint: %s", cudaGetErrorString(e));
  if (rc == EPO_OK) {
    float2* keep = c->d_dz;
    c->d_dz = dz;
    rc = epo_launch_fused(c, lambda, false, false, true);
    c->d_dz = keep;
    c->static_dirty = true;                          // (the launch above was not the loop's: keep the next one serialised)
  }
  if (rc == EPO_OK) rc = epo_launch_finish(c, false, false, false, true, 0);
  if (rc == EPO_OK) rc = epo_joint_gather_gz(c, dz, gz_dev ? g_depth : d_gz);
  bool sync = false;
  if (rc == EPO_OK) {
    epo_launch_f64_to_f32(st, c->d_glogf, d_gf32, (int64_t)N);
    c->launches += 1;
    e = copy_out(g_logf, d_gf32, N * sizeof(float), st, &sync);
    if (e == cudaSuccess && !gz_dev) e = copy_out(g_depth, d_gz, px * sizeof(float), st, &sync);
    if (e == cudaSuccess && loss) {
      epo_launch_f64_to_f32(st, &c->d_state->loss, c->d_out_f, 1);
      c->launches += 1;
      e = copy_out(loss, c->d_out_f, sizeof(float), st, &sync);
    }
    if (e == cudaSuccess && sync) e = cudaStreamSynchronize(st);
    if (e != cudaSuccess) rc = epo_fail(c, EPO_ERR_CUDA, "epo_loss_grad_joint: %s", cudaGetErrorString(e));
  }
  epo_dfree(c, d_gf32); epo_dfree(c, d_gz); epo_dfree(c, dz_tmp);
  return rc;
}

epo_status epo_get_joint_variables(epo_ctx* c, double* gamma, double* alpha, double* beta) {
  if (!c) return EPO_ERR_INVALID_ARG;
  if (!c->have_views || !c->cfg.joint_phase) return epo_fail(c, EPO_ERR_BAD_STATE, "epo_get_joint_variables needs cfg.joint_phase and epo_set_views");
  if ((alpha == nullptr) != (beta == nullptr)) return epo_fail(c, EPO_ERR_INVALID_ARG, "epo_get_joint_variables: alpha and beta come together");
  EPO_CUDA(c, cudaSetDevice(c->cfg.device));
  cudaStream_t st = c->stream;
  const size_t N = (size_t)c->N, px = N * c->W * c->H;
  double *d_a = nullptr, *d_b = nullptr;
  const bool maps = alpha != nullptr, dev = maps && is_device_ptr(alpha) && is_device_ptr(beta);
  cudaError_t e = cudaSuccess;
  if (maps && !dev) { e = epo_dmalloc(c, &d_a, px * sizeof(double)); if (e == cudaSuccess) e = epo_dmalloc(c, &d_b, px * sizeof(double)); }
  epo_status rc = e == cudaSuccess ? epo_joint_export(c, nullptr, maps ? (dev ? alpha : d_a) : nullptr, maps ? (dev ? beta : d_b) : nullptr)
                                   : epo_fail(c, EPO_ERR_OUT_OF_MEMORY, "epo_get_joint_variables: %s", cudaGetErrorString(e));
  bool sync = false;
  if (rc == EPO_OK && gamma) e = copy_out(gamma, c->d_gamma, N * sizeof(double), st, &sync);
  if (rc == EPO_OK && e == cudaSuccess && maps && !dev) {
    e = copy_out(alpha, d_a, px * sizeof(double), st, &sync);
    if (e == cudaSuccess) e = copy_out(beta, d_b, px * sizeof(double), st, &sync);
  }
  if (e == cudaSuccess && sync) e = cudaStreamSynchronize(st);
  if (rc == EPO_OK && e != cudaSuccess) rc = epo_fail(c, EPO_ERR_CUDA, "epo_get_joint_variables: %s", cudaGetErrorString(e));
  epo_dfree(c, d_a); epo_dfree(c, d_b);
  return rc;
}

epo_status epo_step(epo_ctx* c, int32_t n_iters, int32_t* iters_done, int32_t* phase) {
  if (!c) return EPO_ERR_INVALID_ARG;
  NvtxRange nvtx_("epo: epo_step");
  if (!c->have_views || !c->have_pairs) return epo_fail(c, EPO_ERR_BAD_STATE, "epo_step before epo_set_views/epo_set_pairs");
  if (n_iters < 0) return epo_fail(c, EPO_ERR_INVALID_ARG, "epo_step: negative iteration count");
  EPO_CUDA(c, cudaSetDevice(c->cfg.device));
  cudaStream_t st = c->stream;
  // Whole bodies of the loop graph (graph_unroll iterations each) run as ONE launch that loops on the device until
  // they are used up or the rule stops the loop; the remainder (and short calls) is enqueued kernel by kernel.  After a
  // stop at most one body's and one remainder's worth of iterations is launched in vain (their kernels exit at once).
  const int in_graph = c->use_graph ? n_iters / c->graph_unroll * c->graph_unroll : 0;
  if (in_graph > 0 && !c->step_exec) EPO_TRY(build_step_graph(c));
  if (in_graph > 0 && c->step_exec) {
    EpoBeginArgs ba;
    epo_begin_step_call_args(c, n_iters, in_graph, c->step_cond, &ba);
    cudaKernelNodeParams kp = {};
    kp.func = ba.func; kp.gridDim = dim3(1); kp.blockDim = dim3(1); kp.sharedMemBytes = 0; kp.kernelParams = ba.ptrs; kp.extra = nullptr;
    EPO_CUDA(c, cudaGraphExecKernelNodeSetParams(c->step_exec, c->step_begin_node, &kp));
    EPO_CUDA(c, cudaGraphLaunch(c->step_exec, st));
    c->static_dirty = false;
    // kernels these iterations run if no rule stops them (what the host loop would have launched)
    c->launches += 1 + (int64_t)in_graph * (2 + (c->subsample ? 1 : 0) + (c->cfg.joint_phase ? 1 : 0));
    for (int i = in_graph; i < n_iters; ++i) EPO_TRY(enqueue_iteration(c, 0));
  } else if (n_iters == 0) {
    EPO_TRY(epo_launch_begin_step_call(c, 0));
  } else {
    // no k_begin_step_call: the first iteration's kernels gate on DevState.stopped and its k_finish opens the call
    // (iters_done, budget, halt); one launch less per call, which is what a step-by-step caller pays per iteration
    for (int i = 0; i < n_iters; ++i) {
      c->first_budget = i == 0 ? n_iters : 0;
      const epo_status rc = enqueue_iteration(c, 0);
      c->first_budget = 0;
      if (rc != EPO_OK) return rc;
    }
  }
  // joint loop: the iterations just enqueued rewrite K (k_finish) and the packed points (k_joint_points, which signals
  // programmatic completion at its top).  A fused launch that reads them BEFORE its dependency wait -- every non-joint
  // one, e.g. the next epo_loss_grad -- must therefore not overlap them: keep it serialised.  Joint fused launches read
  // after the wait and ignore the flag.
  if (c->cfg.joint_phase && n_iters > 0) c->static_dirty = true;
  bool sync = false;
  if (iters_done) EPO_CUDA(c, copy_out(iters_done, &c->d_state->iters_done, sizeof(int32_t), st, &sync));
  if (phase) EPO_CUDA(c, copy_out(phase, &c->d_state->phase, sizeof(int32_t), st, &sync));
  if (sync) EPO_CUDA(c, cudaStreamSynchronize(st));
  return EPO_OK;
}

epo_status epo_get_poses_f64(epo_ctx* c, double* poses) {
  if (!c) return EPO_ERR_INVALID_ARG;
  if (!c->have_views) return epo_fail(c, EPO_ERR_BAD_STATE, "epo_get_poses before epo_set_views");
  if (!poses) return epo_fail(c, EPO_ERR_INVALID_ARG, "epo_get_poses: NULL output");
  EPO_CUDA(c, cudaSetDevice(c->cfg.device));
  bool sync = false;
  EPO_CUDA(c, copy_out(poses, c->d_poses, (size_t)c->N * 12 * sizeof(double), c->stream, &sync));
  if (sync) EPO_CUDA(c, cudaStreamSynchronize(c->stream));
  return EPO_OK;
}

epo_status epo_get_poses(epo_ctx* c, float* poses) {
  if (!c) return EPO_ERR_INVALID_ARG;
  NvtxRange nvtx_("epo: epo_get_poses");
  if (!c->have_views) return epo_fail(c, EPO_ERR_BAD_STATE, "epo_get_poses before epo_set_views");
  if (!poses) return epo_fail(c, EPO_ERR_INVALID_ARG, "epo_get_poses: NULL output");
  EPO_CUDA(c, cudaSetDevice(c->cfg.device));
  cudaStream_t st = c->stream;
  const int64_t n = (int64_t)c->N * 12;
  if (is_device_ptr(poses)) {
    epo_launch_f64_to_f32(st, c->d_poses, poses, n);
    c->launches += 1;
    EPO_CUDA(c, cudaGetLastError());
    return EPO_OK;
  }
  float* tmp = nullptr;
  EPO_CUDA(c, epo_dmalloc(c, &tmp, (size_t)n * sizeof(float)));
  epo_launch_f64_to_f32(st, c->d_poses, tmp, n);
  c->launches += 1;
  cudaError_t e = cudaMemcpyAsync(poses, tmp, (size_t)n * sizeof(float), cudaMemcpyDeviceToHost, st);
  if (e == cudaSuccess) e = cudaStreamSynchronize(st);
  epo_dfree(c, tmp);
  if (e != cudaSuccess) return epo_fail(c, EPO_ERR_CUDA, "epo_get_poses: %s", cudaGetErrorString(e));
  return EPO_OK;
}

epo_status epo_reset(epo_ctx* c, const float* poses) {
  if (!c) return EPO_ERR_INVALID_ARG;
  NvtxRange nvtx_("epo: epo_reset");
  if (!c->have_views) return epo_fail(c, EPO_ERR_BAD_STATE, "epo_reset before epo_set_views");
  EPO_CUDA(c, cudaSetDevice(c->cfg.device));
  cudaStream_t st = c->stream;
  const size_t n = (size_t)c->N * 12;
  if (poses) {
    std::vector<float> hP(n);
    EPO_CUDA(c, cudaMemcpyAsync(hP.data(), poses, n * sizeof(float), cudaMemcpyDefault, st));
    EPO_CUDA(c, cudaStreamSynchronize(st));
    for (size_t k = 0; k < n; ++k)
      if (!std::isfinite(hP[k])) return epo_fail(c, EPO_ERR_INVALID_ARG, "epo_reset: non-finite pose");
    float* tmp = nullptr;
    EPO_CUDA(c, epo_dmalloc(c, &tmp, n * sizeof(float)));
    cudaError_t e = cudaMemcpyAsync(tmp, hP.data(), n * sizeof(float), cudaMemcpyHostToDevice, st);
    if (e == cudaSuccess) { epo_launch_f32_to_f64(st, tmp, c->d_poses_init, (int64_t)n); c->launches += 1; e = cudaStreamSynchronize(st); }
    epo_dfree(c, tmp);
    if (e != cudaSuccess) return epo_fail(c, EPO_ERR_CUDA, "epo_reset: %s", cudaGetErrorString(e));
  }
  EPO_CUDA(c, cudaMemcpyAsync(c->d_poses, c->d_poses_init, n * sizeof(double), cudaMemcpyDeviceToDevice, st));
  EPO_TRY(reset_optimiser(c));
  return EPO_OK;
}

epo_status epo_get_edge_counts(epo_ctx* c, int32_t* offsets) {
  if (!c) return EPO_ERR_INVALID_ARG;
  if (!c->have_views) return epo_fail(c, EPO_ERR_BAD_STATE, "epo_get_edge_counts before epo_set_views");
  if (!offsets) return epo_fail(c, EPO_ERR_INVALID_ARG, "NULL output");
  EPO_CUDA(c, cudaSetDevice(c->cfg.device));
  bool sync = false;
  EPO_CUDA(c, copy_out(offsets, c->d_edge_off, (size_t)(c->N + 1) * sizeof(int32_t), c->stream, &sync));
  if (sync) EPO_CUDA(c, cudaStreamSynchronize(c->stream));
  return EPO_OK;
}

epo_status epo_get_edge_list(epo_ctx* c, int32_t view, uint16_t* uv, float* z) {
  if (!c) return EPO_ERR_INVALID_ARG;
  if (!c->have_views) return epo_fail(c, EPO_ERR_BAD_STATE, "epo_get_edge_list before epo_set_views");
  if (view < 0 || view >= c->N || !uv || !z) return epo_fail(c, EPO_ERR_INVALID_ARG, "epo_get_edge_list: bad argument");
  EPO_CUDA(c, cudaSetDevice(c->cfg.device));
  const int32_t lo = c->h_edge_off[view], n = c->h_edge_off[view + 1] - lo;
  if (n == 0) return EPO_OK;
  // records are (u | v << 16, z): de-interleave on the host side of the boundary (marshalling only)
  std::vector<EdgeRec> h((size_t)n);
  EPO_CUDA(c, cudaMemcpyAsync(h.data(), c->d_edges + lo, (size_t)n * sizeof(EdgeRec), cudaMemcpyDeviceToHost, c->stream));
  EPO_CUDA(c, cudaStreamSynchronize(c->stream));
  std::vector<uint16_t> huv((size_t)n * 2); std::vector<float> hz((size_t)n);
  for (int32_t i = 0; i < n; ++i) { huv[2 * i] = (uint16_t)(h[i].uv & 0xffffu); huv[2 * i + 1] = (uint16_t)(h[i].uv >> 16); hz[i] = h[i].z; }
  EPO_CUDA(c, cudaMemcpyAsync(uv, huv.data(), (size_t)n * 2 * sizeof(uint16_t), cudaMemcpyDefault, c->stream));
  EPO_CUDA(c, cudaMemcpyAsync(z, hz.data(), (size_t)n * sizeof(float), cudaMemcpyDefault, c->stream));
  EPO_CUDA(c, cudaStreamSynchronize(c->stream));
  return EPO_OK;
}

epo_status epo_get_dtf(epo_ctx* c, int32_t view, float* dtf) {
  if (!c) return EPO_ERR_INVALID_ARG;
  if (!c->have_views) return epo_fail(c, EPO_ERR_BAD_STATE, "epo_get_dtf before epo_set_views");
  if (view < 0 || view >= c->N || !dtf) return epo_fail(c, EPO_ERR_INVALID_ARG, "epo_get_dtf: bad argument");
  EPO_CUDA(c, cudaSetDevice(c->cfg.device));
  // the field lives only in the atlas the kernel samples: read view's tile back (fp16 fields are widened)
  const size_t W = (size_t)c->W, H = (size_t)c->H;
  const size_t ax = (size_t)(view % c->atlas.cols) * W, ay = (size_t)(view / c->atlas.cols) * H;
  if (c->cfg.dtf_format == 1) {
    std::vector<__half> h(W * H);
    EPO_CUDA(c, cudaMemcpy2DFromArrayAsync(h.data(), W * sizeof(__half), c->atlas.arr, ax * sizeof(__half), ay,
                                           W * sizeof(__half), H, cudaMemcpyDeviceToHost, c->stream));
    EPO_CUDA(c, cudaStreamSynchronize(c->stream));
    std::vector<float> f(W * H);
    for (size_t i = 0; i < W * H; ++i) f[i] = __half2float(h[i]);
    EPO_CUDA(c, cudaMemcpyAsync(dtf, f.data(), W * H * sizeof(float), cudaMemcpyDefault, c->stream));
    EPO_CUDA(c, cudaStreamSynchronize(c->stream));
    return EPO_OK;
  }
  const bool dev = is_device_ptr(dtf);
  EPO_CUDA(c, cudaMemcpy2DFromArrayAsync(dtf, W * sizeof(float), c->atlas.arr, ax * sizeof(float), ay, W * sizeof(float), H,
                                         dev ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost, c->stream));
  if (!dev) EPO_CUDA(c, cudaStreamSynchronize(c->stream));
  return EPO_OK;
}

epo_status epo_get_pair_order(epo_ctx* c, int32_t* canonical_pairs, int32_t* perm) {
  if (!c) return EPO_ERR_INVALID_ARG;
  if (!c->have_pairs) return epo_fail(c, EPO_ERR_BAD_STATE, "epo_get_pair_order before epo_set_pairs");
  EPO_CUDA(c, cudaSetDevice(c->cfg.device));
  bool sync = false;
  if (canonical_pairs) EPO_CUDA(c, copy_out(canonical_pairs, c->d_pairs, (size_t)c->P * sizeof(int2), c->stream, &sync));
  if (perm) EPO_CUDA(c, copy_out(perm, c->d_perm, (size_t)c->P * sizeof(int32_t), c->stream, &sync));
  if (sync) EPO_CUDA(c, cudaStreamSynchronize(c->stream));
  return EPO_OK;
}

epo_status epo_get_trace(epo_ctx* c, int32_t first, int32_t count, float* loss, float* theta95) {
  if (!c) return EPO_ERR_INVALID_ARG;
  if (!c->have_pairs) return epo_fail(c, EPO_ERR_BAD_STATE, "epo_get_trace before epo_set_pairs");
  if (first < 0 || count < 0 || first + count > c->cfg.max_steps) return epo_fail(c, EPO_ERR_INVALID_ARG, "epo_get_trace: bad range");
  EPO_CUDA(c, cudaSetDevice(c->cfg.device));
  cudaStream_t st = c->stream;
  bool sync = false;
  if (loss) {
    float* stage = c->d_out_f + 1 + (size_t)c->N * 6 + (size_t)c->P;
    epo_launch_f64_to_f32(st, c->d_loss_trace + first, stage, count);
    EPO_CUDA(c, copy_out(loss, stage, (size_t)count * sizeof(float), st, &sync));
  }
  if (theta95) {
    float* stage = c->d_out_f + 1 + (size_t)c->N * 6 + (size_t)c->P + c->cfg.max_steps;
    epo_launch_f64_to_f32(st, c->d_theta + first, stage, count);
    EPO_CUDA(c, copy_out(theta95, stage, (size_t)count * sizeof(float), st, &sync));
  }
  if (sync) EPO_CUDA(c, cudaStreamSynchronize(st));
  return EPO_OK;
}

epo_status epo_extract_edges(epo_ctx* c, const uint8_t* images, int32_t low, int32_t high, uint8_t* edges) {
  if (!c) return EPO_ERR_INVALID_ARG;
  NvtxRange nvtx_("epo: epo_extract_edges");
  if (!images || !edges || low < 0 || high < low || high > 1442)    // |g| <= 1020 sqrt(2)
    return epo_fail(c, EPO_ERR_INVALID_ARG, "epo_extract_edges: bad argument");
  EPO_CUDA(c, cudaSetDevice(c->cfg.device));
  cudaStream_t st = c->stream;
  const size_t px = (size_t)c->N * c->W * c->H;
  uint8_t *d_img = nullptr, *d_out = nullptr;
  const bool in_dev = is_device_ptr(images), out_dev = is_device_ptr(edges);
  cudaError_t e = cudaSuccess;
  if (!in_dev) { e = epo_dmalloc(c, &d_img, px); if (e == cudaSuccess) e = cudaMemcpyAsync(d_img, images, px, cudaMemcpyHostToDevice, st); }
  if (e == cudaSuccess && !out_dev) e = epo_dmalloc(c, &d_out, px);
  epo_status rc = e == cudaSuccess ? epo_run_canny(c, in_dev ? images : d_img, low, high, out_dev ? edges : d_out)
                                   : epo_fail(c, e == cudaErrorMemoryAllocation ? EPO_ERR_OUT_OF_MEMORY : EPO_ERR_CUDA,
                                              "epo_extract_edges: %s", cudaGetErrorString(e));
  if (rc == EPO_OK && !out_dev) {
    e = cudaMemcpyAsync(edges, d_out, px, cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    if (e != cudaSuccess) rc = epo_fail(c, EPO_ERR_CUDA, "epo_extract_edges: %s", cudaGetErrorString(e));
  }
  epo_dfree(c, d_img); epo_dfree(c, d_out);
  return rc;
}

epo_status epo_extract_edges_rgb(epo_ctx* c, const uint8_t* rgb, int32_t low, int32_t high, uint8_t* edges) {
  if (!c) return EPO_ERR_INVALID_ARG;
  NvtxRange nvtx_("epo: epo_extract_edges_rgb");
  if (!rgb || !edges || low < 0 || high < low || high > 1442)
    return epo_fail(c, EPO_ERR_INVALID_ARG, "epo_extract_edges_rgb: bad argument");
  EPO_CUDA(c, cudaSetDevice(c->cfg.device));
  cudaStream_t st = c->stream;
  const size_t px = (size_t)c->N * c->W * c->H;
  uint8_t *d_rgb = nullptr, *d_grey = nullptr;
  const bool in_dev = is_device_ptr(rgb);
  cudaError_t e = epo_dmalloc(c, &d_grey, px);
  if (e == cudaSuccess && !in_dev) { e = epo_dmalloc(c, &d_rgb, 3 * px); if (e == cudaSuccess) e = cudaMemcpyAsync(d_rgb, rgb, 3 * px, cudaMemcpyHostToDevice, st); }
  epo_status rc = e == cudaSuccess ? epo_run_rgb_to_grey(c, in_dev ? rgb : d_rgb, d_grey)
                                   : epo_fail(c, e == cudaErrorMemoryAllocation ? EPO_ERR_OUT_OF_MEMORY : EPO_ERR_CUDA,
                                              "epo_extract_edges_rgb: %s", cudaGetErrorString(e));
  if (rc == EPO_OK) rc = epo_extract_edges(c, d_grey, low, high, edges);      // device grey in: no further staging
  epo_dfree(c, d_rgb); epo_dfree(c, d_grey);
  return rc;
}

epo_status epo_build_viewgraph(epo_ctx* c, int32_t grid_stride, float tau, float min_frac, int32_t* pairs, int64_t capacity,
                               int64_t* n_pairs, int32_t* counts) {
  if (!c) return EPO_ERR_INVALID_ARG;
  NvtxRange nvtx_("epo: epo_build_viewgraph");
  if (!c->have_views) return epo_fail(c, EPO_ERR_BAD_STATE, "epo_build_viewgraph before epo_set_views");
  if (!n_pairs || grid_stride < 1 || !(tau > 0.f) || !(min_frac >= 0.f && min_frac <= 1.f) || capacity < 0 || (capacity > 0 && !pairs))
    return epo_fail(c, EPO_ERR_INVALID_ARG, "epo_build_viewgraph: bad argument");
  EPO_CUDA(c, cudaSetDevice(c->cfg.device));
  cudaStream_t st = c->stream;
  const size_t N = (size_t)c->N;
  int2 *d_counts = nullptr, *d_pairs = nullptr; long long* d_n = nullptr;
  cudaError_t e = epo_dmalloc(c, &d_counts, N * N * sizeof(int2));
  if (e == cudaSuccess) e = epo_dmalloc(c, &d_pairs, (N * (N - 1) + 1) * sizeof(int2));
  if (e == cudaSuccess) e = epo_dmalloc(c, &d_n, sizeof(long long));
  epo_status rc = e == cudaSuccess ? epo_launch_viewgraph(c, grid_stride, tau, min_frac, d_counts, d_pairs, d_n)
                                   : epo_fail(c, e == cudaErrorMemoryAllocation ? EPO_ERR_OUT_OF_MEMORY : EPO_ERR_CUDA,
                                              "epo_build_viewgraph: %s", cudaGetErrorString(e));
  long long n = 0;
  if (rc == EPO_OK) {
    e = cudaMemcpyAsync(&n, d_n, sizeof(long long), cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    if (e != cudaSuccess) rc = epo_fail(c, EPO_ERR_CUDA, "epo_build_viewgraph: %s", cudaGetErrorString(e));
  }
  if (rc == EPO_OK) {
    *n_pairs = n;
    if (pairs && n > capacity) rc = epo_fail(c, EPO_ERR_INVALID_ARG, "epo_build_viewgraph: %lld pairs do not fit a capacity of %lld", n, (long long)capacity);
  }
  if (rc == EPO_OK && pairs && n > 0) {
    e = cudaMemcpyAsync(pairs, d_pairs, (size_t)n * sizeof(int2), cudaMemcpyDefault, st);
    if (e != cudaSuccess) rc = epo_fail(c, EPO_ERR_CUDA, "epo_build_viewgraph: %s", cudaGetErrorString(e));
  }
  if (rc == EPO_OK && counts) {
    e = cudaMemcpyAsync(counts, d_counts, N * N * sizeof(int2), cudaMemcpyDefault, st);
    if (e != cudaSuccess) rc = epo_fail(c, EPO_ERR_CUDA, "epo_build_viewgraph: %s", cudaGetErrorString(e));
  }
  cudaStreamSynchronize(st);
  epo_dfree(c, d_counts); epo_dfree(c, d_pairs); epo_dfree(c, d_n);
  return rc;
}

epo_status epo_get_pair_subset(epo_ctx* c, int32_t step, uint8_t* flags) {
  if (!c) return EPO_ERR_INVALID_ARG;
  if (!c->have_pairs) return epo_fail(c, EPO_ERR_BAD_STATE, "epo_get_pair_subset before epo_set_pairs");
  if (!flags || step < 0) return epo_fail(c, EPO_ERR_INVALID_ARG, "epo_get_pair_subset: bad argument");
  EPO_CUDA(c, cudaSetDevice(c->cfg.device));
  cudaStream_t st = c->stream;
  std::vector<uint8_t> h((size_t)c->P, 1), out((size_t)c->P, 1);
  if (c->subsample) {
    // the kernel of the loop, at the given step, flags only; then canonical -> caller's order (marshalling)
    EPO_TRY(epo_launch_select_pairs(c, step, false, false));
    std::vector<int32_t> perm((size_t)c->P);
    EPO_CUDA(c, cudaMemcpyAsync(h.data(), c->d_sel_flag, (size_t)c->P, cudaMemcpyDeviceToHost, st));
    EPO_CUDA(c, cudaMemcpyAsync(perm.data(), c->d_perm, (size_t)c->P * sizeof(int32_t), cudaMemcpyDeviceToHost, st));
    EPO_CUDA(c, cudaStreamSynchronize(st));
    for (int64_t q = 0; q < c->P; ++q) out[(size_t)perm[(size_t)q]] = h[(size_t)q];
  }
  EPO_CUDA(c, cudaMemcpyAsync(flags, out.data(), (size_t)c->P, cudaMemcpyDefault, st));
  EPO_CUDA(c, cudaStreamSynchronize(st));
  return EPO_OK;
}

static epo_status time_fused(epo_ctx* c, float lambda, int32_t reps, int32_t flush_l2, float* ms_mean, float* ms_min,
                             bool gather_only);

epo_status epo_time_loss_grad_kernel(epo_ctx* c, float lambda, int32_t reps, int32_t flush_l2, float* ms_mean,
                                     float* ms_min) {
  return time_fused(c, lambda, reps, flush_l2, ms_mean, ms_min, false);
}

epo_status epo_time_gather_ceiling(epo_ctx* c, float lambda, int32_t reps, int32_t flush_l2, float* ms_mean,
                                   float* ms_min) {
  return time_fused(c, lambda, reps, flush_l2, ms_mean, ms_min, true);
}

static epo_status time_fused(epo_ctx* c, float lambda, int32_t reps, int32_t flush_l2, float* ms_mean, float* ms_min,
                             bool gather_only) {
  if (!c) return EPO_ERR_INVALID_ARG;
  if (!c->have_views || !c->have_pairs) return epo_fail(c, EPO_ERR_BAD_STATE, "epo_time_loss_grad_kernel before set_views/set_pairs");
  if (reps < 1 || !(lambda >= 0.f)) return epo_fail(c, EPO_ERR_INVALID_ARG, "epo_time_loss_grad_kernel: bad argument");
  if (gather_only) {
    // the recorded taps are 16-bit atlas coordinates (x | y << 16, all ones = "not valid"): refuse atlases they cannot hold
    const int64_t aw = (int64_t)c->atlas.cols * c->W, ah = (int64_t)((c->N + c->atlas.cols - 1) / c->atlas.cols) * c->H;
    if (aw > 65535 || ah > 65535)
      return epo_fail(c, EPO_ERR_UNSUPPORTED, "epo_time_gather_ceiling: atlas of %lld x %lld texels exceeds the 16-bit tap record",
                      (long long)aw, (long long)ah);
  }
  EPO_CUDA(c, cudaSetDevice(c->cfg.device));
  cudaStream_t st = c->stream;
  const size_t flush_bytes = (size_t)256 << 20;   // > 126 MB L2
  void* flush = nullptr;
  uint2* taps = nullptr; unsigned* gout = nullptr;
  cudaEvent_t e0 = nullptr, e1 = nullptr;
  if (flush_l2) EPO_CUDA(c, epo_dmalloc(c, &flush, flush_bytes));
  cudaError_t e = cudaEventCreate(&e0);
  if (e == cudaSuccess) e = cudaEventCreate(&e1);
  epo_status rc = EPO_OK;
  const size_t n_items = (size_t)(c->n_work > 0 ? c->n_work : 1);
  if (gather_only && e == cudaSuccess) {
    // the tap stream of this evaluation, recorded once by the fused kernel's own position arithmetic
    e = epo_dmalloc(c, &taps, n_items * (size_t)(c->lg_chunk / 2) * sizeof(uint2));
    if (e == cudaSuccess) e = epo_dmalloc(c, &gout, n_items * sizeof(unsigned));
    if (e == cudaSuccess) e = cudaMemsetAsync(gout, 0, n_items * sizeof(unsigned), st);
    if (e == cudaSuccess) rc = epo_launch_record_taps(c, lambda, taps);
  }
  double sum = 0.0; float mn = 1e30f;
  for (int r = 0; r < reps && e == cudaSuccess && rc == EPO_OK; ++r) {
    if (flush) e = cudaMemsetAsync(flush, r & 0xff, flush_bytes, st);
    if (e == cudaSuccess) e = cudaEventRecord(e0, st);
    if (e == cudaSuccess) rc = gather_only ? epo_launch_gather_taps(c, lambda, taps, gout) : epo_launch_fused_only(c, lambda);
    if (e == cudaSuccess) e = cudaEventRecord(e1, st);
    if (e == cudaSuccess) e = cudaEventSynchronize(e1);
    float ms = 0.f;
    if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, e0, e1);
    sum += ms; if (ms < mn) mn = ms;
  }
  if (e == cudaSuccess) e = cudaStreamSynchronize(st);
  epo_dfree(c, flush); epo_dfree(c, taps); epo_dfree(c, gout);
  if (e0) cudaEventDestroy(e0);
  if (e1) cudaEventDestroy(e1);
  if (rc != EPO_OK) return rc;
  if (e != cudaSuccess) return epo_fail(c, e == cudaErrorMemoryAllocation ? EPO_ERR_OUT_OF_MEMORY : EPO_ERR_CUDA, "epo_time_loss_grad_kernel: %s", cudaGetErrorString(e));
  if (ms_mean) *ms_mean = (float)(sum / reps);
  if (ms_min) *ms_min = mn;
  return EPO_OK;
}

// ---- optimiser state export / import (SURVEY.md section 5 "checkpoint / resume") -----------------------------------------
// Everything epo_step changes, as one flat blob: header | poses | Adam m | Adam v | DevState | theta trace | loss trace
// [ | gamma + AdamW moments | K | depth_stepped | (alpha, beta) | their moments | packed points ]  (joint contexts).
// Views, fields, pair lists and work lists are NOT in it: they are functions of the inputs the caller still has.
namespace {
struct StateHeader {
  uint64_t magic;                 // "EPOSTATE"
  int32_t version, n_views, width, height, max_steps, joint;
  int64_t n_pairs, n_edges, n_slots, bytes;
};
constexpr uint64_t kStateMagic = 0x4554415453'4f5045ull;   // 'E' 'P' 'O' 'S' 'T' 'A' 'T' 'E' little-endian
struct StateSeg { void* p; size_t bytes; };

size_t state_align(size_t b) { return (b + 15) & ~(size_t)15; }

std::vector<StateSeg> state_segments(epo_ctx* c) {
  const size_t N = (size_t)c->N, T = (size_t)c->cfg.max_steps;
  std::vector<StateSeg> v = {{c->d_poses, N * 12 * sizeof(double)}, {c->d_m, N * 6 * sizeof(double)}, {c->d_v, N * 6 * sizeof(double)},
                             {c->d_state, sizeof(DevState)}, {c->d_theta, T * sizeof(double)}, {c->d_loss_trace, T * sizeof(double)}};
  if (c->cfg.joint_phase) {
    const size_t S = c->packed.h_off.empty() ? 0 : (size_t)c->packed.h_off[c->N] / 2;
    v.push_back({c->d_gamma, 3 * N * sizeof(double)});
    v.push_back({c->d_K, N * 4 * sizeof(float)});
    v.push_back({c->d_depth_stepped, sizeof(int32_t)});
    if (S > 0) {
      v.push_back({c->d_ab, S * sizeof(double4)});
      v.push_back({c->d_abm, 2 * S * sizeof(float4)});
      v.push_back({c->packed.xyz, S * 3 * sizeof(float2)});
    }
  }
  return v;
}

StateHeader state_header(epo_ctx* c) {
  StateHeader h = {};
  h.magic = kStateMagic; h.version = 1; h.n_views = c->N; h.width = c->W; h.height = c->H; h.max_steps = c->cfg.max_steps;
  h.joint = c->cfg.joint_phase; h.n_pairs = c->P; h.n_edges = c->E;
  h.n_slots = c->packed.h_off.empty() ? 0 : (int64_t)c->packed.h_off[c->N] / 2;
  size_t b = state_align(sizeof(StateHeader));
  for (const StateSeg& sg : state_segments(c)) b += state_align(sg.bytes);
  h.bytes = (int64_t)b;
  return h;
}
}  // namespace

epo_status epo_get_state_size(epo_ctx* c, int64_t* bytes) {
  if (!c) return EPO_ERR_INVALID_ARG;
  if (!bytes) return epo_fail(c, EPO_ERR_INVALID_ARG, "epo_get_state_size: NULL output");
  if (!c->have_views || !c->have_pairs) return epo_fail(c, EPO_ERR_BAD_STATE, "epo_get_state_size before epo_set_views/epo_set_pairs");
  *bytes = state_header(c).bytes;
  return EPO_OK;
}

epo_status epo_get_state(epo_ctx* c, void* blob, int64_t capacity) {
  if (!c) return EPO_ERR_INVALID_ARG;
  if (!c->have_views || !c->have_pairs) return epo_fail(c, EPO_ERR_BAD_STATE, "epo_get_state before epo_set_views/epo_set_pairs");
  const StateHeader h = state_header(c);
  if (!blob || capacity < h.bytes) return epo_fail(c, EPO_ERR_INVALID_ARG, "epo_get_state: need %lld bytes, got %lld", (long long)h.bytes, (long long)capacity);
  EPO_CUDA(c, cudaSetDevice(c->cfg.device));
  cudaStream_t st = c->stream;
  char* out = static_cast<char*>(blob);
  EPO_CUDA(c, cudaMemcpyAsync(out, &h, sizeof(h), cudaMemcpyDefault, st));
  size_t off = state_align(sizeof(StateHeader));
  for (const StateSeg& sg : state_segments(c)) {
    EPO_CUDA(c, cudaMemcpyAsync(out + off, sg.p, sg.bytes, cudaMemcpyDefault, st));
    off += state_align(sg.bytes);
  }
  EPO_CUDA(c, cudaStreamSynchronize(st));              // the header is copied from this frame
  return EPO_OK;
}

epo_status epo_set_state(epo_ctx* c, const void* blob, int64_t bytes) {
  if (!c) return EPO_ERR_INVALID_ARG;
  if (!c->have_views || !c->have_pairs) return epo_fail(c, EPO_ERR_BAD_STATE, "epo_set_state before epo_set_views/epo_set_pairs");
  if (!blob || bytes < (int64_t)sizeof(StateHeader)) return epo_fail(c, EPO_ERR_INVALID_ARG, "epo_set_state: blob too short");
  EPO_CUDA(c, cudaSetDevice(c->cfg.device));
  cudaStream_t st = c->stream;
  StateHeader got;
  EPO_CUDA(c, cudaMemcpyAsync(&got, blob, sizeof(got), cudaMemcpyDefault, st));
  EPO_CUDA(c, cudaStreamSynchronize(st));
  const StateHeader want = state_header(c);
  if (got.magic != kStateMagic || got.version != want.version)
    return epo_fail(c, EPO_ERR_INVALID_ARG, "epo_set_state: not a state blob of this library version");
  if (got.n_views != want.n_views || got.width != want.width || got.height != want.height || got.max_steps != want.max_steps ||
      got.joint != want.joint || got.n_pairs != want.n_pairs || got.n_edges != want.n_edges || got.n_slots != want.n_slots ||
      got.bytes != want.bytes || bytes < want.bytes)
    return epo_fail(c, EPO_ERR_INVALID_ARG, "epo_set_state: the blob was taken from a different problem or configuration "
                    "(views %d/%d, %dx%d/%dx%d, max_steps %d/%d, joint %d/%d, pairs %lld/%lld, edge pixels %lld/%lld, bytes %lld/%lld)",
                    got.n_views, want.n_views, got.width, got.height, want.width, want.height, got.max_steps, want.max_steps,
                    got.joint, want.joint, (long long)got.n_pairs, (long long)want.n_pairs, (long long)got.n_edges,
                    (long long)want.n_edges, (long long)got.bytes, (long long)want.bytes);
  const char* in = static_cast<const char*>(blob);
  size_t off = state_align(sizeof(StateHeader));
  for (const StateSeg& sg : state_segments(c)) {
    EPO_CUDA(c, cudaMemcpyAsync(sg.p, in + off, sg.bytes, cudaMemcpyDefault, st));
    off += state_align(sg.bytes);
  }
  c->static_dirty = true;                               // K / points may have changed under the next fused launch
  EPO_CUDA(c, cudaStreamSynchronize(st));              // the caller may free the blob on return
  return EPO_OK;
}

epo_status epo_get_work(epo_ctx* c, int64_t* reprojections_per_eval, int64_t* kernel_launches_so_far) {
  if (!c) return EPO_ERR_INVALID_ARG;
  if (reprojections_per_eval) *reprojections_per_eval = c->have_pairs ? c->reproj_per_eval : 0;
  if (kernel_launches_so_far) *kernel_launches_so_far = c->launches;
  return EPO_OK;
}

}  // extern "C"
