// ckf.cu — C ABI of the B200-native CKF track-finding library (include/ckf.h): host side.
//
// ckf_create uploads the geometry store (a1) and field store (a2) once and reserves every
// workspace; ckf_find enqueues its launches (four small kernels per level) on the caller's stream and never allocates.
// There is no CPU path in this library: all arithmetic of the method runs in the kernels of
// ckf_step.cuh / ckf_visit.cuh / ckf_branch.cuh / ckf_sort.cuh / ckf_emit.cuh.
#include <cuda_runtime.h>

#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <atomic>
#include <deque>
#include <mutex>
#include <string>
#include <vector>

#include "../../include/ckf.h"
#include "ckf_emit.cuh"
#include "ckf_host_geom.h"
#include "ckf_branch.cuh"
#include "ckf_fit.cuh"
#include "ckf_peak.cuh"
#include "ckf_resolve.cuh"
#include "ckf_seed.cuh"
#include "ckf_sort.cuh"
#include "ckf_step.cuh"
#include "ckf_visit.cuh"

using namespace ckf;

// Scratch of ckf_resolve_static (include/ckf.h): rank keys [MAX_TRACKS] u64 | minima [2][MAX_MEASUREMENTS] u64 |
// owners [MAX_MEASUREMENTS] i32 | states [MAX_TRACKS] i32 | 4 counters.  On the host this NAME is a stand-in, not a
// device address: the entry point takes the address with cudaGetSymbolAddress, once per device.
static __device__ __align__(256) unsigned char g_resolve_static_scratch[CKF_RESOLVE_STATIC_SCRATCH_BYTES];

namespace {

// Error text is per calling THREAD (several host threads may drive one handle, configs[4]): a failing call stores its
// message here and ckf_last_error returns the calling thread's last message.
thread_local std::string g_error;

struct Workspace {
  // link buffer
  double* lk_x = nullptr;
  void* lk_C = nullptr;
  int32_t *lk_module = nullptr, *lk_parent = nullptr, *lk_meas = nullptr, *lk_counts = nullptr, *lk_lastmeas = nullptr;
  void *lk_chi2 = nullptr, *lk_chi2sum = nullptr;
  int32_t *sd = nullptr;       // 3 * max_seeds + 2 * (max_seeds + 1)
  int32_t* seed_tile = nullptr;  // 2 * (tiles + 1)
  int32_t* leaf = nullptr;     // 3 * max_seeds * cap
  // level state (tips, move state, predictions, selections, scan)
  int32_t *tip_link = nullptr, *tip_seed = nullptr;
  double *mv_y = nullptr, *pd_x = nullptr;
  void *mv_D = nullptr, *mv_Dr = nullptr, *mv_dep = nullptr, *pd_C = nullptr, *sel_chi2 = nullptr;
  int32_t *mv_from = nullptr, *mv_tgt = nullptr, *mv_stop = nullptr, *sel_idx = nullptr, *mv_order = nullptr;
  int32_t *t_nsel = nullptr, *t_want = nullptr, *t_counts = nullptr, *t_keep = nullptr, *t_kex = nullptr, *blk_sum = nullptr, *t_fin = nullptr;
  void *s_loc = nullptr, *s_var = nullptr, *s_v0max = nullptr;  // gate index (ckf_sort_slices)
  int32_t* s_idx = nullptr;
  int32_t* globals = nullptr;  // GlobalId
  unsigned long long* counters = nullptr;
  // staging for ckf_find_host
  int32_t* h_moff = nullptr; void *h_loc = nullptr, *h_var = nullptr;
  int32_t* h_smod = nullptr; void *h_sx = nullptr, *h_sC = nullptr;
  int32_t *o_nt = nullptr, *o_off = nullptr, *o_meas = nullptr, *o_seed = nullptr, *o_nh = nullptr, *o_lm = nullptr,
          *o_stop = nullptr;
  void *o_par = nullptr, *o_cov = nullptr, *o_c2 = nullptr, *o_ec2 = nullptr;
  int32_t* pinned_nt = nullptr;  // host pinned [3]: candidates, status, entries of the last ckf_find_host
  cudaEvent_t done = nullptr;    // recorded after the last piece of work that uses this workspace
  // Ownership.  `stream_tag` / `used` (which stream's finds map to this workspace) change under the handle mutex;
  // `busy` is held by a host thread from before its first enqueue to after it has recorded `done`, so a thread that
  // recycles the workspace for another stream waits (on the host) until the previous owner has finished ENQUEUING and
  // then (on the device, cudaStreamWaitEvent) until that work has finished RUNNING.  `done_stream` is written under busy.
  std::mutex busy;
  std::atomic<void*> done_stream{nullptr};
  std::atomic<bool> done_valid{false};
  std::atomic<bool> enqueuing{false};  // a host thread is between acquire_ws and release_ws (hint for others_in_flight)
  void* stream_tag = nullptr;
  bool used = false;
  float last_ms[10] = {0};  // per-kernel-kind times of the last timed ckf_find (ckf_set_timing)
  int last_launches = 0;
  // CUDA graph of the last repeated find on this workspace (launch_find): its key = the kernel parameters + launch policy
  cudaGraphExec_t graph_exec = nullptr;
  cudaStream_t cap_stream = nullptr;
  std::vector<unsigned char> graph_key, last_key;
};

}  // namespace

struct ckf_handle {
  ckf_config cfg;
  int device = 0, sm_count = 0;
  int n_modules = 0, n_layers = 0;
  ModuleRec* d_mod = nullptr;
  LayerRec* d_layer = nullptr;
  GeoDev geo;   // device pointers + layer summary (barrel count, first discs)
  float* d_grid = nullptr;
  FieldDev fld;
  CfgDev kcfg;
  int step_grid = 0, step_regs = 0, visit_grid = 0, visit_smem = 0, tcap = 0, tsize = 4;
  std::deque<Workspace> ws;
  int next_ws = 0;
  std::mutex mu;
  std::vector<void*> allocs;
  // sizes of the last ckf_find_host result, the guess for the next call's device->host copies
  std::atomic<int> hint_tracks{-1}, hint_entries{-1};
  // state store of ckf_fit, reserved in ckf_create (config.max_fit_tracks)
  double* fs_x = nullptr; void* fs_t = nullptr; int32_t* fs_meas = nullptr; int32_t* fs_next = nullptr;
  // level arrays, globals and counters for ckf_step when it runs the moves of a fit level (tcap = fit_chunk)
  int32_t* ft_g = nullptr; unsigned long long* ft_counters = nullptr;
  double* ft_y = nullptr; void *ft_D = nullptr, *ft_Dr = nullptr, *ft_dep = nullptr;
  int32_t *ft_from = nullptr, *ft_tgt = nullptr, *ft_stop = nullptr, *ft_order = nullptr;
  int fit_chunk = 0, fit_states = 0;
  cudaEvent_t fit_done = nullptr;
  // workspace of ckf_resolve (one per handle; calls are ordered one after the other)
  unsigned long long *rs_key = nullptr, *rs_best = nullptr;
  int32_t *rs_owner = nullptr, *rs_state = nullptr, *rs_g = nullptr;
  int resolve_grid = 0;
  cudaEvent_t resolve_done = nullptr;
  // workspace of ckf_seed (one per handle; reserved when config.max_seed_doublets > 0)
  double *sd_sp = nullptr, *sd_cot = nullptr;
  int32_t *sd_cnt = nullptr, *sd_off = nullptr, *sd_t = nullptr, *sd_g = nullptr;
  cudaEvent_t seed_done = nullptr;
  bool timing_print = false;
  // which kernels of a find are launched with overlap (launch_chain): bit 1 sort, 2 step, 4 visit, 8 scan, 16 update,
  // 32 emission, 64 ckf_fit_level.  Measured (profiles/r02_launch_overlap.md): step + visit + update is best; with ckf_scan in the chain as
  // well the whole level loop is one cascade of waiting blocks and a batched find gets 10 % slower.  CKF_CHAIN_OVERLAP=<mask>
  // overrides (0 = plain launches), for A/B measurements.
  bool use_graph = false;  // CKF_GRAPH=1: replay a find that repeats the previous call's arguments from a CUDA graph (opt-in:
                           // capturing and instantiating the graph allocates, which ckf_find otherwise never does)
  bool grad = false;  // J2': config.field_gradient on an interpolated field (a uniform field has no gradient: the default kernels)
  int chain_overlap = 2 | 4 | 16 | 64;
  bool timing = false;  // ckf_set_timing / CKF_TIMING=1: per-kernel CUDA-event times of every ckf_find on stderr (debug aid; synchronises)
};

namespace {

int fail(ckf_handle* h, int code, const char* fmt, ...) {
  char buf[512];
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(buf, sizeof(buf), fmt, ap);
  va_end(ap);
  (void)h;
  g_error = buf;
  return code;
}

#define CK(call)                                                                                        \
  do {                                                                                                  \
    cudaError_t e_ = (call);                                                                            \
    if (e_ != cudaSuccess) return fail(h, CKF_E_CUDA, "%s failed: %s", #call, cudaGetErrorString(e_)); \
  } while (0)

template <typename P>
cudaError_t dalloc(ckf_handle* h, P** p, size_t bytes) {
  void* q = nullptr;
  cudaError_t e = cudaMalloc(&q, bytes ? bytes : 16);
  if (e == cudaSuccess) { h->allocs.push_back(q); *p = (P*)q; }
  return e;
}

// Resident blocks per SM ckf_step / ckf_visit are compiled for: 3 x 128 threads at <= 168 registers (float step:
// measured faster than 4 x 128 at 128 registers with 300 B of spills), 3 x 128 at <= 168 registers (float visit: its
// arrival algebra is float64 since r02; 4 blocks spill 360 B and run 3 % slower, 2 blocks 2 % slower),
// 2 x 128 threads at <= 255 registers (double: the covariance algebra doubles its register footprint).
#ifndef CKF_MINB
#define CKF_MINB 3
#endif
template <typename T> struct MinBlocks { static constexpr int value = CKF_MINB; };
template <> struct MinBlocks<double> { static constexpr int value = 2; };
#ifndef CKF_VISIT_MINB
#define CKF_VISIT_MINB 3
#endif
template <typename T> struct VisitBlocks { static constexpr int value = CKF_VISIT_MINB; };
template <> struct VisitBlocks<double> { static constexpr int value = 2; };

template <typename T>
void fill_params(ckf_handle* h, Workspace& w, KParams<T>& p) {
  const ckf_config& c = h->cfg;
  p.geo = h->geo;
  p.fld = h->fld;
  p.cfg = h->kcfg;
  p.max_links = c.max_links;
  p.lk_x = w.lk_x; p.lk_C = (double*)w.lk_C; p.lk_module = w.lk_module; p.lk_parent = w.lk_parent; p.lk_meas = w.lk_meas;
  p.lk_chi2 = (T*)w.lk_chi2; p.lk_chi2sum = (double*)w.lk_chi2sum; p.lk_counts = w.lk_counts; p.lk_lastmeas = w.lk_lastmeas;
  const size_t S = (size_t)c.max_seeds;
  p.sd_extra = w.sd; p.sd_nemit = w.sd + S; p.sd_nentries = w.sd + 2 * S;
  p.sd_track_base = w.sd + 3 * S; p.sd_entry_base = w.sd + 3 * S + (S + 1);
  p.sd_eoff = w.sd + 3 * S + 2 * (S + 1);
  p.seed_tile = w.seed_tile; p.seed_tiles_cap = (int32_t)((S + SEED_TILE - 1) / SEED_TILE);
  const size_t LC = S * (size_t)c.max_candidates_per_seed;
  p.leaf_link = w.leaf; p.leaf_meta = w.leaf + LC; p.leaf_entry = w.leaf + 2 * LC;
  p.tcap = h->tcap;
  p.tip_link = w.tip_link; p.tip_seed = w.tip_seed;
  p.mv_y = w.mv_y; p.mv_D = (T*)w.mv_D; p.mv_Dr = (T*)w.mv_Dr; p.mv_dep = (double*)w.mv_dep; p.mv_from = w.mv_from; p.mv_tgt = w.mv_tgt;
  p.mv_stop = w.mv_stop; p.mv_order = w.mv_order;
  p.pd_x = w.pd_x; p.pd_C = (double*)w.pd_C; p.sel_chi2 = (T*)w.sel_chi2; p.sel_idx = w.sel_idx;
  p.t_nsel = w.t_nsel; p.t_want = w.t_want; p.t_counts = w.t_counts; p.t_keep = w.t_keep; p.t_kex = w.t_kex;
  p.blk_sum = w.blk_sum; p.t_fin = w.t_fin;
  p.s_loc = (typename Vec2<T>::type*)w.s_loc; p.s_var = (typename Vec2<T>::type*)w.s_var; p.s_idx = w.s_idx;
  p.s_v0max = (T*)w.s_v0max;
  p.g = w.globals;
  p.counters = w.counters;
  p.max_tracks = c.max_tracks; p.max_entries = c.max_track_entries;
  p.o_summary = nullptr;
}

// ckf_step with the gradient terms (J2') carries 27 + 12 more live numbers: two resident blocks per SM instead of three.
template <typename T, bool GRAD> struct StepBlocks { static constexpr int value = GRAD ? 2 : MinBlocks<T>::value; };

// Launch configuration: ckf_step is persistent (one wave of resident blocks), ckf_visit grid-strides.
template <typename T, bool GRAD>
int setup_launch(ckf_handle* h, const ckf_config* c) {
  int per_sm = 0, vper_sm = 0;
  cudaFuncAttributes fa;
  auto step = ckf_step<T, StepBlocks<T, GRAD>::value, GRAD>;
  auto visit = ckf_visit<T, VisitBlocks<T>::value, GRAD>;
  h->visit_smem = (int)((VISIT_NT / 32) * VSmem<T>::bytes(c->max_branches_per_surface));
  if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, step, STEP_NT, 0) != cudaSuccess ||
      cudaFuncGetAttributes(&fa, step) != cudaSuccess ||
      cudaFuncSetAttribute(visit, cudaFuncAttributeMaxDynamicSharedMemorySize, h->visit_smem) != cudaSuccess ||
      cudaOccupancyMaxActiveBlocksPerMultiprocessor(&vper_sm, visit, VISIT_NT, h->visit_smem) != cudaSuccess)
    return fail(h, CKF_E_CUDA, "launch configuration failed: %s", cudaGetErrorString(cudaGetLastError()));
  if (per_sm < 1 || vper_sm < 1) return fail(h, CKF_E_CUDA, "kernels do not fit on an SM (visit smem %d B)", h->visit_smem);
  h->step_regs = fa.numRegs;
  h->step_grid = per_sm * h->sm_count;
  h->visit_grid = vper_sm * h->sm_count;
  return CKF_OK;
}

// One kernel of a find's chain.  With `overlap` the launch carries programmatic stream serialisation: the kernel's blocks
// become resident while the previous kernel of the stream drains and wait in chain_enter() for its completion, which
// takes the launch latency out of the ~136 dependent launches of a find.
template <typename... KArgs, typename... Args>
void launch_chain(void (*kernel)(KArgs...), int grid, int block, size_t smem, cudaStream_t st, bool overlap, Args&&... args) {
  cudaLaunchConfig_t lc = {};
  lc.gridDim = dim3((unsigned)grid); lc.blockDim = dim3((unsigned)block); lc.dynamicSmemBytes = smem; lc.stream = st;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  at[0].val.programmaticStreamSerializationAllowed = 1;
  lc.attrs = at; lc.numAttrs = overlap ? 1 : 0;
  cudaLaunchKernelEx(&lc, kernel, KArgs(args)...);
}

// Is a find of this handle being enqueued or still running on ANOTHER stream (work of `st` itself is ordered before
// whatever is enqueued next, never beside it)?  A hint, read without locks: it only selects the launch policy.
bool others_in_flight(ckf_handle* h, const Workspace* self, cudaStream_t st) {
  for (auto& o : h->ws) {
    if (&o == self) continue;
    if (o.enqueuing.load()) return true;
    if (o.done_valid.load() && o.done_stream.load() != (void*)st && cudaEventQuery(o.done) != cudaSuccess) {
      (void)cudaGetLastError();  // 'not ready' is an answer, not an error of this call; any other answer (an event of a
      return true;               // capturing stream, say) is taken the careful way: plain launches
    }
  }
  return false;
}

template <typename T>
int launch_find(ckf_handle* h, Workspace& w, const ckf_measurements* m, const ckf_seeds* s, ckf_tracks* o,
                cudaStream_t st, int32_t* summary = nullptr) {
  KParams<T> p;
  std::memset(&p, 0, sizeof(p));   // padding too: the bytes of p are the key of the graph cache below
  fill_params<T>(h, w, p);
  p.o_summary = summary;
  p.n_meas = m->n; p.n_seeds = s->n;
  p.moff = m->module_offsets;
  p.n_vmod = std::max(1, m->n_events) * h->n_modules;
  p.loc = (const typename Vec2<T>::type*)m->loc;
  p.var = (const typename Vec2<T>::type*)m->var;
  p.seed_module = s->module_id; p.seed_x = (const T*)s->params; p.seed_C = (const T*)s->cov;
  p.o_ntracks = o->n_tracks; p.o_status = o->status; p.o_offsets = o->track_offsets; p.o_meas = o->meas_idx;
  p.o_seed = o->seed_id; p.o_nholes = o->n_holes; p.o_lastmod = o->last_module; p.o_stop = o->stop_reason;
  p.o_params = (T*)o->params; p.o_cov = (T*)o->cov; p.o_chi2sum = (T*)o->chi2_sum; p.o_entrychi2 = (T*)o->entry_chi2;
  const int nb = (std::max(s->n, (int)CNT_N) + 255) / 256;
  // optional per-kernel timing (debug): an event after every launch
  std::vector<cudaEvent_t> tev;
  std::vector<int> tkind;
  auto mark = [&](int kind) {
    if (!h->timing) return;
    cudaEvent_t e;
    cudaEventCreate(&e);
    cudaEventRecord(e, st);
    tev.push_back(e);
    tkind.push_back(kind);
  };
  mark(-1);
  // Launch policy.  Alone on the GPU a find is a chain of ~70 short dependent kernels and overlapped launches take the
  // launch latency out of it (3.70 -> 3.45 ms).  With other finds in flight the SMs are shared, blocks that sit resident
  // waiting for their predecessor take room from the other streams' kernels (2 batches in flight: 20.4 -> 19.2 M
  // seeds/s), so the launches stay plain.  Timing mode puts an event between the kernels, which serialises them anyway.
  const int ovm = (h->timing || others_in_flight(h, &w, st)) ? 0 : h->chain_overlap;
  auto enqueue = [&](cudaStream_t q) {
    ckf_init_event<T><<<nb, 256, 0, q>>>(p); mark(0);  // plain launch: whatever precedes the find in the stream is not ours
    launch_chain(ckf_sort_slices<T>, h->sm_count * (1024 / SORT_NT), SORT_NT, 0, q, ovm & 1, p); mark(1);
    // level loop: tips of level l were made by level l - 1; a tip at max_levels only stops (LEVEL_LIMIT) and emits.
    // Kernels of an empty level return at once, so the loop needs no host read of the level's size.
    const int wide = h->sm_count * 4;
    for (int level = 0; level <= h->cfg.max_levels; ++level) {
      if (h->grad) {
        if (level > 0) { launch_chain(ckf_step<T, StepBlocks<T, true>::value, true>, h->step_grid, STEP_NT, 0, q, ovm & 2, p, level); mark(2); }
        launch_chain(ckf_visit<T, VisitBlocks<T>::value, true>, h->visit_grid, VISIT_NT, h->visit_smem, q, ovm & 4, p, level); mark(3);
      } else {
        if (level > 0) { launch_chain(ckf_step<T, MinBlocks<T>::value>, h->step_grid, STEP_NT, 0, q, ovm & 2, p, level); mark(2); }
        launch_chain(ckf_visit<T, VisitBlocks<T>::value>, h->visit_grid, VISIT_NT, h->visit_smem, q, ovm & 4, p, level); mark(3);
      }
      launch_chain(ckf_scan<T>, wide, SCAN_NT, 0, q, ovm & 8, p, level); mark(5);
      launch_chain(ckf_update<T>, wide, SCAN_NT, 0, q, ovm & 16, p, level); mark(6);
    }
    launch_chain(ckf_scan_seeds<T>, (s->n + SEED_TILE - 1) / SEED_TILE + 1, SEED_TILE, 0, q, ovm & 32, p); mark(7);
    launch_chain(ckf_emit_tracks<T>, h->sm_count * 8, EMIT_NT, 0, q, ovm & 32, p); mark(8);
    launch_chain(ckf_finalize<T>, 1, 1, 0, q, ovm & 32, p); mark(9);
  };
  // Opt-in (CKF_GRAPH=1): a find whose arguments repeat (same arrays, same sizes, same launch policy: a pipeline that runs
  // on preallocated, padded buffers) is replayed from a CUDA graph of its ~136 launches: the second call in a row with the same
  // arguments captures it, later ones launch it (configs[3] 3.29 -> 3.20 ms, configs[0] 0.92 -> 0.81 ms).  Anything else
  // -- new arguments, timing mode, a caller who is capturing the stream himself -- is enqueued launch by launch as before.
  bool done = false;
  if (!h->timing && h->use_graph) {
    std::vector<unsigned char> key(sizeof(p) + sizeof(int));
    std::memcpy(key.data(), &p, sizeof(p));
    std::memcpy(key.data() + sizeof(p), &ovm, sizeof(int));
    cudaStreamCaptureStatus cs = cudaStreamCaptureStatusNone;
    if (cudaStreamIsCapturing(st, &cs) != cudaSuccess) { (void)cudaGetLastError(); cs = cudaStreamCaptureStatusActive; }
    if (cs == cudaStreamCaptureStatusNone) {
      if (w.graph_exec && w.graph_key == key) {
        done = cudaGraphLaunch(w.graph_exec, st) == cudaSuccess;
      } else if (w.last_key == key) {
        cudaGraph_t g = nullptr;
        cudaGraphExec_t ge = nullptr;
        // captured on a stream of the workspace's own (the caller's may be the legacy default stream, which cannot
        // capture); the graph does not remember it
        if (!w.cap_stream) cudaStreamCreateWithFlags(&w.cap_stream, cudaStreamNonBlocking);
        if (w.cap_stream && cudaStreamBeginCapture(w.cap_stream, cudaStreamCaptureModeThreadLocal) == cudaSuccess) {
          enqueue(w.cap_stream);
          if (cudaStreamEndCapture(w.cap_stream, &g) == cudaSuccess && g && cudaGraphInstantiate(&ge, g, 0) == cudaSuccess) {
            if (w.graph_exec) cudaGraphExecDestroy(w.graph_exec);
            w.graph_exec = ge;
            w.graph_key = key;
            done = cudaGraphLaunch(w.graph_exec, st) == cudaSuccess;
          }
          if (g) cudaGraphDestroy(g);
        }
        if (!done) (void)cudaGetLastError();   // no graph then: the plain path below
      }
    }
    if (!done) w.last_key.swap(key);
  }
  if (!done) enqueue(st);
  w.last_launches = 5 + 4 * (h->cfg.max_levels + 1) - 1;
  if (h->timing) {
    static const char* names[10] = {"init", "sort", "step", "visit", "cap", "scan", "update", "scan_seeds", "emit", "finalize"};
    cudaStreamSynchronize(st);
    float acc[10] = {0}, tot = 0.f;
    for (size_t i = 1; i < tev.size(); ++i) {
      float ms = 0.f;
      cudaEventElapsedTime(&ms, tev[i - 1], tev[i]);
      acc[tkind[i]] += ms;
      tot += ms;
    }
    for (int k = 0; k < 10; ++k) w.last_ms[k] = acc[k];
    if (h->timing_print) {
      fprintf(stderr, "[ckf timing] total %.3f ms:", tot);
      for (int k = 0; k < 10; ++k) fprintf(stderr, " %s %.3f", names[k], acc[k]);
      fprintf(stderr, "\n");
    }
    for (auto e : tev) cudaEventDestroy(e);
  }
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return fail(h, CKF_E_CUDA, "kernel launch failed: %s", cudaGetErrorString(e));
  return CKF_OK;
}

template <typename T>
int launch_fit(ckf_handle* h, const ckf_measurements* m, const ckf_seeds* s, const ckf_tracks* t, ckf_fits* o,
               cudaStream_t st) {
  FitParams<T> p;
  p.geo = h->geo;
  p.fld = h->fld;
  p.cfg = h->kcfg;
  p.moff = m->module_offsets;
  p.loc = (const typename Vec2<T>::type*)m->loc;
  p.var = (const typename Vec2<T>::type*)m->var;
  p.seed_module = s->module_id; p.seed_x = (const T*)s->params; p.seed_C = (const T*)s->cov;
  p.n_tracks = t->n_tracks; p.offsets = t->track_offsets; p.meas = t->meas_idx; p.seed = t->seed_id;
  p.max_tracks = h->cfg.max_tracks;
  p.chunk = h->fit_chunk; p.max_states = h->fit_states;
  p.fs_x = h->fs_x; p.fs_t = (T*)h->fs_t; p.fs_meas = h->fs_meas; p.fs_next = h->fs_next;
  p.o_status = o->status; p.o_nstates = o->n_states; p.o_chi2 = (T*)o->chi2_sum; p.o_lastx = (T*)o->last_params;
  p.o_lastC = (T*)o->last_cov; p.o_firstC = (T*)o->first_cov; p.o_entryx = (T*)o->entry_params;
  p.o_work = (unsigned long long*)o->work;
  const int grid = (h->fit_chunk + FIT_NT - 1) / FIT_NT;
  // passes of fit_chunk tracks; a pass beyond *n_tracks returns at once (the count is only known on the device)
  // what ckf_step needs to run the moves of one level with one tip per track
  KParams<T> kp;
  std::memset(&kp, 0, sizeof(kp));
  kp.geo = p.geo; kp.fld = p.fld; kp.cfg = p.cfg;
  kp.tcap = h->fit_chunk;
  kp.g = h->ft_g; kp.counters = h->ft_counters;
  kp.mv_y = h->ft_y; kp.mv_D = (T*)h->ft_D; kp.mv_Dr = (T*)h->ft_Dr; kp.mv_dep = (double*)h->ft_dep; kp.mv_from = h->ft_from; kp.mv_tgt = h->ft_tgt;
  kp.mv_stop = h->ft_stop; kp.mv_order = h->ft_order;
  const int n_upper = o->n_tracks_upper > 0 ? std::min(o->n_tracks_upper, h->cfg.max_tracks) : h->cfg.max_tracks;
  const int ovm = others_in_flight(h, nullptr, st) ? 0 : h->chain_overlap;  // launch policy as in launch_find
  for (int first = 0; first < n_upper; first += h->fit_chunk) {
    p.first = first;
    // forward filter, level-synchronous: per level the moves on ckf_step, then the rest of the state (ckf_fit_level).
    // Two blocks of globals, by level parity: level L's ckf_step reads the schedule in block L & 1.
    cudaMemsetAsync(h->ft_g, 0, 2 * GBLK * 4, st);
    cudaMemsetAsync(h->ft_g + G_NTIPS0, 1, 2 * 4, st);       // non-zero: ckf_step only asks whether the level holds tips
    cudaMemsetAsync(h->ft_g + GBLK + G_NTIPS0, 1, 2 * 4, st);
    cudaMemsetAsync(h->ft_counters, 0, CNT_N * 8, st);
    for (int level = 0; level < h->fit_states; ++level) {
      int32_t* g_this = h->ft_g + GBLK * (level & 1);
      int32_t* g_next = h->ft_g + GBLK * ((level + 1) & 1);
      if (level > 0) {
        kp.g = g_this;
        if (h->grad) launch_chain(ckf_step<T, StepBlocks<T, true>::value, true>, h->step_grid, STEP_NT, 0, st, ovm & 2, kp, level);
        else launch_chain(ckf_step<T, MinBlocks<T>::value>, h->step_grid, STEP_NT, 0, st, ovm & 2, kp, level);
      }
      kp.g = g_next;
      if (h->grad) launch_chain(ckf_fit_level<T, true>, grid, FIT_NT, 0, st, ovm & 64, kp, p, level, g_this);
      else launch_chain(ckf_fit_level<T>, grid, FIT_NT, 0, st, ovm & 64, kp, p, level, g_this);
    }
    ckf_fit_flush_work<<<1, 32, 0, st>>>(h->ft_counters, p.o_work);
    const bool f32 = sizeof(T) == 4 && o->smoother_precision == 32;
    if (o->smoother == 1) {
      if (f32) ckf_fit_smooth_tf<T, float><<<grid, FIT_NT, 0, st>>>(p);
      else ckf_fit_smooth_tf<T, double><<<grid, FIT_NT, 0, st>>>(p);
    } else {
      if (f32) ckf_fit_smooth<T, float><<<grid, FIT_NT, 0, st>>>(p);
      else ckf_fit_smooth<T, double><<<grid, FIT_NT, 0, st>>>(p);
    }
  }
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return fail(h, CKF_E_CUDA, "kernel launch failed: %s", cudaGetErrorString(e));
  return CKF_OK;
}

// Picks (or recycles) the workspace for this stream and returns it with `busy` LOCKED; the stream is ordered after the
// workspace's previous work when that ran on another stream.  The caller enqueues, then calls release_ws, which
// records `done` and unlocks -- on every exit path (WsGuard).
Workspace* acquire_ws(ckf_handle* h, cudaStream_t st) {
  Workspace* w = nullptr;
  {
    std::lock_guard<std::mutex> lk(h->mu);
    for (auto& x : h->ws)
      if (x.used && x.stream_tag == (void*)st) { w = &x; break; }
    if (!w)
      for (auto& x : h->ws)
        if (!x.used) { w = &x; break; }
    if (!w) { w = &h->ws[h->next_ws]; h->next_ws = (h->next_ws + 1) % (int)h->ws.size(); }
    w->used = true;
    w->stream_tag = (void*)st;
  }
  w->busy.lock();  // a previous owner still enqueuing: wait for it (and for its cudaEventRecord) on the host
  w->enqueuing = true;
  if (w->done_valid && w->done_stream != (void*)st) cudaStreamWaitEvent(st, w->done, 0);
  return w;
}

void release_ws(Workspace* w, cudaStream_t st) {
  cudaEventRecord(w->done, st);
  w->done_stream = (void*)st;
  w->done_valid = true;
  w->enqueuing = false;
  w->busy.unlock();
}

struct WsGuard {
  Workspace* w; cudaStream_t st;
  ~WsGuard() { release_ws(w, st); }
};

template <typename T>
int launch_seed(ckf_handle* h, const ckf_measurements* m, const ckf_seeding* sc, ckf_seed_out* o, cudaStream_t st) {
  SeedParams<T> p;
  p.geo = h->geo; p.fld = h->fld;
  p.cfg.layer_b = sc->layer_b; p.cfg.layer_m = sc->layer_m; p.cfg.layer_t = sc->layer_t;
  p.cfg.dphi_max = sc->dphi_max; p.cfg.cot_max = sc->cot_max; p.cfg.z0_max = sc->z0_max; p.cfg.dcot_max = sc->dcot_max;
  p.cfg.pt_min = sc->pt_min; p.cfg.d0_max = sc->d0_max; p.cfg.sigma_angle = sc->sigma_angle;
  p.cfg.rel_sigma_qop = sc->rel_sigma_qop; p.cfg.cov_scale = sc->cov_scale;
  p.n_meas = m->n; p.moff = m->module_offsets; p.loc = (const T*)m->loc; p.var = (const T*)m->var;
  p.sp = h->sd_sp; p.n_cap = h->cfg.max_measurements; p.cnt = h->sd_cnt; p.mt_off = h->sd_off; p.mt_t = h->sd_t;
  p.mt_cot = h->sd_cot; p.max_doublets = h->cfg.max_seed_doublets; p.g = h->sd_g;
  p.capacity = o->capacity; p.o_n = o->n_seeds; p.o_status = o->status; p.o_module = o->module_id;
  p.o_params = (T*)o->params; p.o_cov = (T*)o->cov; p.o_triplets = o->triplets;
  const int wide = h->sm_count * 8, n = m->n;
  seed_spacepoints<T><<<wide, 128, 0, st>>>(p);
  cudaMemsetAsync(p.cnt, 0, ((size_t)n + 1) * 4, st);
  seed_doublets_mt<T, false><<<wide, 128, 0, st>>>(p);
  seed_scan<<<1, 1024, 0, st>>>(p.cnt, p.mt_off, n, p.g + 0);
  seed_doublets_mt<T, true><<<wide, 128, 0, st>>>(p);
  cudaMemsetAsync(p.cnt, 0, ((size_t)n + 1) * 4, st);
  seed_triplets<T, false><<<wide, 128, 0, st>>>(p);
  seed_scan<<<1, 1024, 0, st>>>(p.cnt, p.cnt, n, p.g + 1);
  seed_triplets<T, true><<<wide, 128, 0, st>>>(p);
  seed_finish<T><<<1, 1, 0, st>>>(p);
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return fail(h, CKF_E_CUDA, "ckf_seed launch failed: %s", cudaGetErrorString(e));
  return CKF_OK;
}

}  // namespace

extern "C" {

int ckf_abi_version(void) { return CKF_ABI_VERSION; }

const char* ckf_last_error(const ckf_handle* h) { (void)h; return g_error.c_str(); }

int ckf_create(const ckf_geometry* g, const ckf_field* f, const ckf_config* c, ckf_handle** out) {
  ckf_handle* h = nullptr;
  if (!g || !f || !c || !out) return fail(h, CKF_E_ARG, "null argument");
  *out = nullptr;
  if (c->precision != 32 && c->precision != 64) return fail(h, CKF_E_ARG, "precision must be 32 or 64");
  if (c->max_branches_per_surface < 1 || c->max_branches_per_surface > 32)
    return fail(h, CKF_E_ARG, "max_branches_per_surface must be in 1..32");
  if (c->max_candidates_per_seed < 1 || c->max_candidates_per_seed > 256)
    return fail(h, CKF_E_ARG, "max_candidates_per_seed must be in 1..256");
  if (c->max_levels < 1 || c->max_levels > 64) return fail(h, CKF_E_ARG, "max_levels must be in 1..64");
  if (c->min_measurements < 1) return fail(h, CKF_E_ARG, "min_measurements must be >= 1");
  if (c->max_seeds < 1 || c->max_measurements < 0 || c->max_tracks < 1 || c->max_track_entries < 1 || c->n_streams < 1 ||
      c->max_fit_tracks < 0 || c->max_seed_doublets < 0)
    return fail(h, CKF_E_ARG, "capacities must be positive");
  if (g->n_layers < 1 || g->n_modules < 1) return fail(h, CKF_E_ARG, "empty geometry");
  if (g->n_layers > 254) return fail(h, CKF_E_ARG, "at most 254 layers (the navigation cursors are 9-bit fields)");
  if (f->kind != 0 && f->kind != 1) return fail(h, CKF_E_ARG, "field kind must be 0 or 1");
  if (c->field_gradient != 0 && c->field_gradient != 1) return fail(h, CKF_E_ARG, "field_gradient must be 0 or 1");
  if (f->kind == 1 && (!f->grid || f->n[0] < 2 || f->n[1] < 2 || f->n[2] < 2))
    return fail(h, CKF_E_ARG, "field grid needs >= 2 nodes per axis");
  for (int l = 0; l < g->n_layers; ++l)
    if (g->n_phi[l] < 3 || g->n_z[l] < 1) return fail(h, CKF_E_ARG, "layer %d: n_phi >= 3 and n_z >= 1 required", l);
  if (g->layer_kind) {   // row f3: barrel layers first, by increasing radius, then the discs
    bool disc_seen = false;
    for (int l = 0; l < g->n_layers; ++l) {
      const int k = g->layer_kind[l];
      if (k != 0 && k != 1) return fail(h, CKF_E_ARG, "layer %d: kind must be 0 (barrel) or 1 (disc)", l);
      if (k == 1) disc_seen = true;
      else if (disc_seen) return fail(h, CKF_E_ARG, "barrel layers must precede the disc layers");
      if (k == 1 && (!g->layer_r_min || !(g->layer_r_min[l] >= 0.0) || !(g->layer_r_min[l] < g->layer_r[l]) || g->layer_half_z[l] == 0.0))
        return fail(h, CKF_E_ARG, "disc layer %d: needs 0 <= r_min < r and a plane z != 0", l);
    }
  }
  for (int l = 1; l < g->n_layers; ++l)
    if ((!g->layer_kind || (g->layer_kind[l] == 0 && g->layer_kind[l - 1] == 0)) && !(g->layer_r[l] > g->layer_r[l - 1]))
      return fail(h, CKF_E_ARG, "barrel layer radii must increase");
  if (g->layer_kind && g->layer_kind[0] != 0) return fail(h, CKF_E_ARG, "the first layer must be a barrel layer");

  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1)
    return fail(h, CKF_E_CUDA, "no CUDA device: this library has no CPU fallback");
  h = new ckf_handle();
  h->cfg = *c;
  if (h->cfg.max_events_per_find <= 0) h->cfg.max_events_per_find = 1;
  if (h->cfg.max_links <= 0) h->cfg.max_links = (int32_t)std::min<long long>(48LL * c->max_seeds, 0x7ffffff0LL);
  h->tsize = c->precision == 32 ? 4 : 8;
  auto bail = [&](int code) { std::string e = g_error; ckf_destroy(h); g_error = e; return code; };
  cudaDeviceProp prop;
  if (cudaGetDevice(&h->device) != cudaSuccess || cudaGetDeviceProperties(&prop, h->device) != cudaSuccess) {
    fail(h, CKF_E_CUDA, "cudaGetDeviceProperties failed");
    return bail(CKF_E_CUDA);
  }
  h->sm_count = prop.multiProcessorCount;
  { const char* t = getenv("CKF_TIMING"); h->timing = h->timing_print = t && t[0] == '1'; }
  { const char* t = getenv("CKF_GRAPH"); h->use_graph = t && t[0] == '1'; }
  { const char* t = getenv("CKF_CHAIN_OVERLAP"); if (t && t[0]) h->chain_overlap = atoi(t); }
  h->n_modules = g->n_modules;
  h->n_layers = g->n_layers;

  // ---- a1 geometry store
  std::vector<ModuleRec> mods;
  std::vector<LayerRec> layers;
  build_geometry_records(*g, mods, layers);
#define CKB(call)                                                                            \
  do {                                                                                       \
    cudaError_t e_ = (call);                                                                 \
    if (e_ != cudaSuccess) {                                                                 \
      fail(h, CKF_E_CUDA, "%s failed: %s", #call, cudaGetErrorString(e_));                   \
      return bail(CKF_E_CUDA);                                                               \
    }                                                                                        \
  } while (0)
  CKB(dalloc(h, &h->d_mod, mods.size() * sizeof(ModuleRec)));
  CKB(dalloc(h, &h->d_layer, layers.size() * sizeof(LayerRec)));
  CKB(cudaMemcpy(h->d_mod, mods.data(), mods.size() * sizeof(ModuleRec), cudaMemcpyHostToDevice));
  CKB(cudaMemcpy(h->d_layer, layers.data(), layers.size() * sizeof(LayerRec), cudaMemcpyHostToDevice));
  h->geo.mod = h->d_mod; h->geo.layer = h->d_layer; h->geo.n_layers = g->n_layers; h->geo.n_modules = g->n_modules;
  fill_geo_summary(layers, h->geo);
  h->geo.bidir = c->bidirectional ? 1 : 0;
  // ---- a2 field store
  std::memset(&h->fld, 0, sizeof(h->fld));
  h->fld.kind = f->kind;
  h->grad = c->field_gradient == 1 && f->kind == 1;
  for (int a = 0; a < 3; ++a) {
    h->fld.ub[a] = f->uniform_b[a];
    h->fld.n[a] = f->n[a];
    h->fld.org[a] = f->origin[a];
    h->fld.inv[a] = f->kind == 1 ? 1.0 / f->spacing[a] : 0.0;
    h->fld.nm2[a] = (double)(f->n[a] - 2);
  }
  {
    // device copy of the grid: entry (i, j, k) = node (i, j, k) and node (i, j, k + 1), 8 float32 (ld_pair); a uniform
    // field still owns a 2 x 2 x 2 grid of its value: field_at never reads it (kind 0 returns first), but ld_pair is a
    // plain asm load which the compiler may hoist above that test, so every address field_at can form must be
    // readable -- with n = 2 the index clamps leave only cell 0
    std::vector<float> pairs;
    if (f->kind == 1) {
      fill_field_pairs(f->grid, f->n, pairs);
    } else {
      const float ub[3] = {(float)f->uniform_b[0], (float)f->uniform_b[1], (float)f->uniform_b[2]};
      float cube[8 * 3];
      for (int i = 0; i < 8; ++i) for (int a = 0; a < 3; ++a) cube[3 * i + a] = ub[a];
      const int32_t n2[3] = {2, 2, 2};
      fill_field_pairs(cube, n2, pairs);
      for (int a = 0; a < 3; ++a) { h->fld.n[a] = 2; h->fld.nm2[a] = 0.0; h->fld.org[a] = 0.0; h->fld.inv[a] = 0.0; }
    }
    CKB(dalloc(h, &h->d_grid, pairs.size() * sizeof(float)));
    CKB(cudaMemcpy(h->d_grid, pairs.data(), pairs.size() * sizeof(float), cudaMemcpyHostToDevice));
    h->fld.grid = h->d_grid;
  }
  // ---- config
  h->kcfg.chi2_max = c->chi2_max; h->kcfg.rk_tol = c->rk_tolerance_mm; h->kcfg.surf_tol = c->surface_tolerance_mm;
  h->kcfg.h_max = c->h_max_mm; h->kcfg.mass = c->particle_mass_gev; h->kcfg.max_branches = c->max_branches_per_surface;
  h->kcfg.max_cands = c->max_candidates_per_seed; h->kcfg.max_holes = c->max_holes; h->kcfg.min_meas = c->min_measurements;
  h->kcfg.max_rk_steps = c->max_rk_steps_per_surface; h->kcfg.max_levels = c->max_levels;
  h->kcfg.energy_loss = c->energy_loss ? 1 : 0;
  h->kcfg.field_gradient = h->grad ? 1 : 0;
  // ---- launch configuration: ckf_step is persistent (one wave of resident blocks), ckf_visit grid-strides
  {
    const int rc = h->grad ? (c->precision == 32 ? setup_launch<float, true>(h, c) : setup_launch<double, true>(h, c))
                           : (c->precision == 32 ? setup_launch<float, false>(h, c) : setup_launch<double, false>(h, c));
    if (rc != CKF_OK) return bail(rc);
  }
  if (h->cfg.max_tips_per_level <= 0)
    h->cfg.max_tips_per_level = (int32_t)std::min<long long>(std::max<long long>(8LL * c->max_seeds, 1024), 0x7ffffff0LL);
  if (h->cfg.max_tips_per_level < c->max_seeds) h->cfg.max_tips_per_level = c->max_seeds;
  h->tcap = h->cfg.max_tips_per_level;
  // ---- workspaces
  const size_t L = (size_t)h->cfg.max_links, S = (size_t)c->max_seeds, ts = (size_t)h->tsize;
  for (int i = 0; i < c->n_streams; ++i) h->ws.emplace_back();
  for (auto& w : h->ws) {
    CKB(dalloc(h, &w.lk_x, 6 * L * sizeof(double)));
    CKB(dalloc(h, (char**)&w.lk_C, 21 * L * sizeof(double)));
    CKB(dalloc(h, &w.lk_module, L * 4)); CKB(dalloc(h, &w.lk_parent, L * 4)); CKB(dalloc(h, &w.lk_meas, L * 4));
    CKB(dalloc(h, &w.lk_counts, L * 4)); CKB(dalloc(h, &w.lk_lastmeas, L * 4));
    CKB(dalloc(h, (char**)&w.lk_chi2, L * ts)); CKB(dalloc(h, (char**)&w.lk_chi2sum, L * sizeof(double)));
    CKB(dalloc(h, &w.sd, (4 * S + 2 * (S + 1)) * 4));
    CKB(dalloc(h, &w.seed_tile, 2 * ((S + SEED_TILE - 1) / SEED_TILE + 2) * 4));
    CKB(dalloc(h, &w.leaf, 3 * S * (size_t)c->max_candidates_per_seed * 4));
    const size_t TC = (size_t)h->tcap, KB = (size_t)c->max_branches_per_surface;
    CKB(dalloc(h, &w.tip_link, 2 * TC * 4)); CKB(dalloc(h, &w.tip_seed, 2 * TC * 4));
    CKB(dalloc(h, &w.mv_y, 8 * TC * sizeof(double))); CKB(dalloc(h, &w.pd_x, 6 * TC * sizeof(double)));
    CKB(dalloc(h, (char**)&w.mv_D, (size_t)MVD * TC * ts)); if (h->grad) CKB(dalloc(h, (char**)&w.mv_Dr, (size_t)12 * TC * ts)); CKB(dalloc(h, (char**)&w.mv_dep, (size_t)NDEP * TC * sizeof(double)));
    CKB(dalloc(h, (char**)&w.pd_C, 21 * TC * sizeof(double))); CKB(dalloc(h, (char**)&w.sel_chi2, KB * TC * ts));
    CKB(dalloc(h, &w.sel_idx, KB * TC * 4));
    CKB(dalloc(h, &w.mv_from, TC * 4)); CKB(dalloc(h, &w.mv_tgt, 2 * TC * 4)); CKB(dalloc(h, &w.mv_stop, TC * 4));
    CKB(dalloc(h, &w.t_nsel, TC * 4)); CKB(dalloc(h, &w.t_want, TC * 4)); CKB(dalloc(h, &w.t_counts, TC * 4));
    CKB(dalloc(h, &w.t_keep, TC * 4)); CKB(dalloc(h, &w.t_kex, TC * 4));
    CKB(dalloc(h, &w.blk_sum, (TC / SCAN_NT + 2) * 4));
    CKB(dalloc(h, &w.t_fin, 4 * TC * 4));
    CKB(dalloc(h, (char**)&w.s_loc, 2 * (size_t)c->max_measurements * ts));
    CKB(dalloc(h, (char**)&w.s_var, 2 * (size_t)c->max_measurements * ts));
    CKB(dalloc(h, &w.s_idx, (size_t)c->max_measurements * 4));
    CKB(dalloc(h, (char**)&w.s_v0max, (size_t)g->n_modules * (size_t)h->cfg.max_events_per_find * ts));
    CKB(dalloc(h, &w.globals, GBLK * 4));
    CKB(cudaMemset(w.globals, 0, GBLK * 4));
    static_assert(G_N <= GBLK, "globals block too small");
    CKB(dalloc(h, &w.mv_order, (size_t)NBIN * TC * 4));
    CKB(dalloc(h, &w.counters, CNT_N * 8));
    CKB(cudaEventCreateWithFlags(&w.done, cudaEventDisableTiming));
    // staging for ckf_find_host
    const size_t M = (size_t)c->max_measurements, NTK = (size_t)c->max_tracks, NE = (size_t)c->max_track_entries;
    CKB(dalloc(h, &w.h_moff, ((size_t)g->n_modules * (size_t)h->cfg.max_events_per_find + 1) * 4));
    CKB(dalloc(h, (char**)&w.h_loc, 2 * M * ts)); CKB(dalloc(h, (char**)&w.h_var, 2 * M * ts));
    CKB(dalloc(h, &w.h_smod, S * 4)); CKB(dalloc(h, (char**)&w.h_sx, 6 * S * ts)); CKB(dalloc(h, (char**)&w.h_sC, 36 * S * ts));
    CKB(dalloc(h, &w.o_nt, 8 * 4)); CKB(dalloc(h, &w.o_off, (NTK + 1) * 4)); CKB(dalloc(h, &w.o_meas, NE * 4));
    CKB(dalloc(h, &w.o_seed, NTK * 4)); CKB(dalloc(h, &w.o_nh, NTK * 4)); CKB(dalloc(h, &w.o_lm, NTK * 4));
    CKB(dalloc(h, &w.o_stop, NTK * 4));
    CKB(dalloc(h, (char**)&w.o_par, 6 * NTK * ts)); CKB(dalloc(h, (char**)&w.o_cov, 36 * NTK * ts));
    CKB(dalloc(h, (char**)&w.o_c2, NTK * ts)); CKB(dalloc(h, (char**)&w.o_ec2, NE * ts));
    CKB(cudaMallocHost((void**)&w.pinned_nt, 4 * 4));
  }
  // ---- state store of ckf_fit (row f1): reserved here, so that ckf_fit allocates nothing
  if (c->max_fit_tracks > 0) {
    const int chunk = std::min(std::min(c->max_fit_tracks, c->max_tracks), (int)FIT_CHUNK), ns = c->max_levels;
    const size_t n = (size_t)ns * (size_t)chunk, CHK = (size_t)chunk;
    CKB(dalloc(h, &h->fs_x, n * FS_X * sizeof(double)));
    CKB(dalloc(h, (char**)&h->fs_t, n * FS_T * ts));
    CKB(dalloc(h, &h->fs_meas, n * 4));
    CKB(dalloc(h, &h->fs_next, CHK * 4));
    CKB(dalloc(h, &h->ft_g, 2 * GBLK * 4)); CKB(dalloc(h, &h->ft_counters, CNT_N * 8));
    CKB(dalloc(h, &h->ft_y, 8 * CHK * sizeof(double)));
    CKB(dalloc(h, (char**)&h->ft_D, (size_t)MVD * CHK * ts)); if (h->grad) CKB(dalloc(h, (char**)&h->ft_Dr, (size_t)12 * CHK * ts)); CKB(dalloc(h, (char**)&h->ft_dep, (size_t)NDEP * CHK * sizeof(double)));
    CKB(dalloc(h, &h->ft_from, CHK * 4)); CKB(dalloc(h, &h->ft_tgt, 2 * CHK * 4)); CKB(dalloc(h, &h->ft_stop, CHK * 4));
    CKB(dalloc(h, &h->ft_order, (size_t)NBIN * CHK * 4));
    CKB(cudaEventCreateWithFlags(&h->fit_done, cudaEventDisableTiming));
    h->fit_chunk = chunk; h->fit_states = ns;
  }
  // ---- workspace of ckf_resolve (row f4): 20 B per measurement + 12 B per candidate
  {
    const size_t M = (size_t)c->max_measurements, NTK = (size_t)c->max_tracks;
    CKB(dalloc(h, &h->rs_key, NTK * 8)); CKB(dalloc(h, &h->rs_best, 2 * M * 8));
    CKB(dalloc(h, &h->rs_owner, M * 4)); CKB(dalloc(h, &h->rs_state, NTK * 4)); CKB(dalloc(h, &h->rs_g, 4 * 4));
    CKB(cudaEventCreateWithFlags(&h->resolve_done, cudaEventDisableTiming));
    int per_sm = 0;
    if (c->precision == 32) CKB(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, ckf_resolve_kernel<float>, RESOLVE_NT, 0));
    else CKB(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, ckf_resolve_kernel<double>, RESOLVE_NT, 0));
    h->resolve_grid = std::max(1, per_sm) * h->sm_count;   // a cooperative launch needs every block resident
  }
  // ---- workspace of ckf_seed (row f4): 48 B per measurement + 12 B per middle-top doublet
  if (c->max_seed_doublets > 0) {
    const size_t M = (size_t)c->max_measurements, D = (size_t)c->max_seed_doublets;
    CKB(dalloc(h, &h->sd_sp, 5 * M * sizeof(double)));
    CKB(dalloc(h, &h->sd_cnt, (M + 1) * 4)); CKB(dalloc(h, &h->sd_off, (M + 1) * 4));
    CKB(dalloc(h, &h->sd_t, D * 4)); CKB(dalloc(h, &h->sd_cot, D * sizeof(double)));
    CKB(dalloc(h, &h->sd_g, 4 * 4));
    CKB(cudaEventCreateWithFlags(&h->seed_done, cudaEventDisableTiming));
  }
#undef CKB
  *out = h;
  return CKF_OK;
}

int ckf_find(ckf_handle* h, const ckf_measurements* m, const ckf_seeds* s, ckf_tracks* o, void* stream) {
  if (!h) return CKF_E_ARG;
  if (!m || !s || !o) return fail(h, CKF_E_ARG, "null argument");
  if (m->n < 0 || s->n < 0) return fail(h, CKF_E_ARG, "negative size");
  if (m->n_events < 0 || m->n_events > h->cfg.max_events_per_find)
    return fail(h, CKF_E_CAPACITY, "n_events %d exceeds max_events_per_find %d", m->n_events, h->cfg.max_events_per_find);
  if (s->n > h->cfg.max_seeds || m->n > h->cfg.max_measurements)
    return fail(h, CKF_E_CAPACITY, "n_seeds %d / n_measurements %d exceed capacity %d / %d", s->n, m->n,
                h->cfg.max_seeds, h->cfg.max_measurements);
  if (!m->module_offsets || (m->n > 0 && (!m->loc || !m->var)) || (s->n > 0 && (!s->module_id || !s->params || !s->cov)))
    return fail(h, CKF_E_ARG, "null input array");
  if (!o->n_tracks || !o->status || !o->track_offsets || !o->meas_idx || !o->seed_id || !o->n_holes || !o->last_module ||
      !o->stop_reason || !o->params || !o->cov || !o->chi2_sum || !o->entry_chi2)
    return fail(h, CKF_E_ARG, "null output array");
  cudaStream_t st = (cudaStream_t)stream;
  WsGuard g{acquire_ws(h, st), st};
  return h->cfg.precision == 32 ? launch_find<float>(h, *g.w, m, s, o, st) : launch_find<double>(h, *g.w, m, s, o, st);
}

int ckf_find_host(ckf_handle* h, const ckf_measurements* m, const ckf_seeds* s, ckf_tracks* o, void* stream) {
  if (!h) return CKF_E_ARG;
  if (!m || !s || !o) return fail(h, CKF_E_ARG, "null argument");
  if (m->n < 0 || s->n < 0 || s->n > h->cfg.max_seeds || m->n > h->cfg.max_measurements)
    return fail(h, CKF_E_CAPACITY, "n_seeds %d / n_measurements %d exceed capacity", s->n, m->n);
  if (m->n_events < 0 || m->n_events > h->cfg.max_events_per_find)
    return fail(h, CKF_E_CAPACITY, "n_events %d exceeds max_events_per_find %d", m->n_events, h->cfg.max_events_per_find);
  if (!m->module_offsets || (m->n > 0 && (!m->loc || !m->var)) || (s->n > 0 && (!s->module_id || !s->params || !s->cov)))
    return fail(h, CKF_E_ARG, "null input array");
  if (!o->n_tracks || !o->status || !o->track_offsets || !o->meas_idx || !o->seed_id || !o->n_holes || !o->last_module ||
      !o->stop_reason || !o->params || !o->cov || !o->chi2_sum || !o->entry_chi2)
    return fail(h, CKF_E_ARG, "null output array");
  cudaStream_t st = (cudaStream_t)stream;
  WsGuard g{acquire_ws(h, st), st};
  Workspace* w = g.w;
  const size_t ts = (size_t)h->tsize;
  CK(cudaMemcpyAsync(w->h_moff, m->module_offsets, ((size_t)h->n_modules * (size_t)std::max(1, m->n_events) + 1) * 4,
                     cudaMemcpyHostToDevice, st));
  CK(cudaMemcpyAsync(w->h_loc, m->loc, 2 * (size_t)m->n * ts, cudaMemcpyHostToDevice, st));
  CK(cudaMemcpyAsync(w->h_var, m->var, 2 * (size_t)m->n * ts, cudaMemcpyHostToDevice, st));
  CK(cudaMemcpyAsync(w->h_smod, s->module_id, (size_t)s->n * 4, cudaMemcpyHostToDevice, st));
  CK(cudaMemcpyAsync(w->h_sx, s->params, 6 * (size_t)s->n * ts, cudaMemcpyHostToDevice, st));
  CK(cudaMemcpyAsync(w->h_sC, s->cov, 36 * (size_t)s->n * ts, cudaMemcpyHostToDevice, st));
  ckf_measurements dm = {m->n, w->h_moff, w->h_loc, w->h_var, m->n_events};
  ckf_seeds ds = {s->n, w->h_smod, w->h_sx, w->h_sC};
  ckf_tracks dt = {w->o_nt, w->o_nt + 1, w->o_off, w->o_meas, w->o_seed, w->o_nh, w->o_lm, w->o_stop,
                   w->o_par, w->o_cov, w->o_c2, w->o_ec2};
  // ckf_finalize leaves (candidates, status, entries) in o_nt[4..6] (o_nt[0], o_nt[1] are *n_tracks and *status)
  int rc = h->cfg.precision == 32 ? launch_find<float>(h, *w, &dm, &ds, &dt, st, w->o_nt + 4)
                                  : launch_find<double>(h, *w, &dm, &ds, &dt, st, w->o_nt + 4);
  if (rc != CKF_OK) return rc;
  CK(cudaMemcpyAsync(w->pinned_nt, w->o_nt + 4, 12, cudaMemcpyDeviceToHost, st));
  // The result sizes are only known on the device.  Instead of stopping the stream to learn them, the copies are
  // issued at once for a GUESS (the sizes of the handle's previous ckf_find_host result + 1/8), the stream is
  // synchronised once, and only a result that outgrew the guess costs a second round for its tail.  The first call on
  // a handle has no guess and takes two rounds.
  auto copy_tracks = [&](size_t t0, size_t t1) -> int {   // per-track arrays, tracks [t0, t1); offsets [t0, t1]
    if (t1 <= t0) return CKF_OK;
    const size_t n = t1 - t0;
    CK(cudaMemcpyAsync(o->track_offsets + t0, w->o_off + t0, (n + 1) * 4, cudaMemcpyDeviceToHost, st));
    CK(cudaMemcpyAsync(o->seed_id + t0, w->o_seed + t0, n * 4, cudaMemcpyDeviceToHost, st));
    CK(cudaMemcpyAsync(o->n_holes + t0, w->o_nh + t0, n * 4, cudaMemcpyDeviceToHost, st));
    CK(cudaMemcpyAsync(o->last_module + t0, w->o_lm + t0, n * 4, cudaMemcpyDeviceToHost, st));
    CK(cudaMemcpyAsync(o->stop_reason + t0, w->o_stop + t0, n * 4, cudaMemcpyDeviceToHost, st));
    CK(cudaMemcpyAsync((char*)o->params + 6 * t0 * ts, (char*)w->o_par + 6 * t0 * ts, 6 * n * ts, cudaMemcpyDeviceToHost, st));
    CK(cudaMemcpyAsync((char*)o->cov + 36 * t0 * ts, (char*)w->o_cov + 36 * t0 * ts, 36 * n * ts, cudaMemcpyDeviceToHost, st));
    CK(cudaMemcpyAsync((char*)o->chi2_sum + t0 * ts, (char*)w->o_c2 + t0 * ts, n * ts, cudaMemcpyDeviceToHost, st));
    return CKF_OK;
  };
  auto copy_entries = [&](size_t e0, size_t e1) -> int {
    if (e1 <= e0) return CKF_OK;
    CK(cudaMemcpyAsync(o->meas_idx + e0, w->o_meas + e0, (e1 - e0) * 4, cudaMemcpyDeviceToHost, st));
    CK(cudaMemcpyAsync((char*)o->entry_chi2 + e0 * ts, (char*)w->o_ec2 + e0 * ts, (e1 - e0) * ts, cudaMemcpyDeviceToHost, st));
    return CKF_OK;
  };
  size_t gt = 0, ge = 0;
  const int ht = h->hint_tracks.load(), he = h->hint_entries.load();
  if (ht >= 0) {
    gt = std::min<size_t>((size_t)h->cfg.max_tracks, (size_t)ht + (size_t)ht / 8 + 256);
    ge = std::min<size_t>((size_t)h->cfg.max_track_entries, (size_t)he + (size_t)he / 8 + 4096);
    if ((rc = copy_tracks(0, gt)) != CKF_OK || (rc = copy_entries(0, ge)) != CKF_OK) return rc;
  }
  CK(cudaStreamSynchronize(st));
  const size_t nt = (size_t)w->pinned_nt[0], ne = (size_t)w->pinned_nt[2];
  *o->n_tracks = w->pinned_nt[0];
  *o->status = w->pinned_nt[1];
  if (nt > gt || ne > ge) {
    if ((rc = copy_tracks(gt, nt)) != CKF_OK || (rc = copy_entries(ge, ne)) != CKF_OK) return rc;
    CK(cudaStreamSynchronize(st));
  }
  if (nt == 0) o->track_offsets[0] = 0;
  h->hint_tracks.store((int)nt);
  h->hint_entries.store((int)ne);
  return CKF_OK;
}

int ckf_fit(ckf_handle* h, const ckf_measurements* m, const ckf_seeds* s, const ckf_tracks* t, ckf_fits* o, void* stream) {
  if (!h) return CKF_E_ARG;
  if (!m || !s || !t || !o) return fail(h, CKF_E_ARG, "null argument");
  if (!m->module_offsets || !t->n_tracks || !t->track_offsets || !t->meas_idx || !t->seed_id)
    return fail(h, CKF_E_ARG, "null input array");
  if (o->smoother_precision != 0 && o->smoother_precision != 32 && o->smoother_precision != 64)
    return fail(h, CKF_E_ARG, "smoother_precision must be 0, 32 or 64");
  if (o->smoother != 0 && o->smoother != 1) return fail(h, CKF_E_ARG, "smoother must be 0 (RTS) or 1 (two-filter)");
  if (o->smoother_precision == 32 && h->cfg.precision != 32)
    return fail(h, CKF_E_ARG, "smoother_precision 32 needs a handle of precision 32");
  if (!o->status || !o->n_states || !o->chi2_sum || !o->last_params || !o->last_cov || !o->first_cov || !o->entry_params)
    return fail(h, CKF_E_ARG, "null output array");
  if ((m->n > 0 && (!m->loc || !m->var)) || (s->n > 0 && (!s->module_id || !s->params || !s->cov)))
    return fail(h, CKF_E_ARG, "null input array");
  if (!h->fs_x) return fail(h, CKF_E_CAPACITY, "ckf_fit needs a state store: create the handle with max_fit_tracks > 0");
  cudaStream_t st = (cudaStream_t)stream;
  std::lock_guard<std::mutex> lk(h->mu);
  cudaStreamWaitEvent(st, h->fit_done, 0);  // one state store: fits are ordered one after the other
  int rc = h->cfg.precision == 32 ? launch_fit<float>(h, m, s, t, o, st) : launch_fit<double>(h, m, s, t, o, st);
  cudaEventRecord(h->fit_done, st);
  return rc;
}

int ckf_seed(ckf_handle* h, const ckf_measurements* m, const ckf_seeding* sc, ckf_seed_out* o, void* stream) {
  if (!h) return CKF_E_ARG;
  if (!m || !sc || !o) return fail(h, CKF_E_ARG, "null argument");
  if (!h->sd_sp) return fail(h, CKF_E_CAPACITY, "ckf_seed needs its workspace: create the handle with max_seed_doublets > 0");
  if (m->n < 0 || m->n > h->cfg.max_measurements) return fail(h, CKF_E_CAPACITY, "n_measurements %d exceeds capacity", m->n);
  if (m->n_events > 1) return fail(h, CKF_E_ARG, "ckf_seed takes one event at a time");
  if (!m->module_offsets || (m->n > 0 && (!m->loc || !m->var))) return fail(h, CKF_E_ARG, "null input array");
  if (!o->n_seeds || !o->status || !o->module_id || !o->params || !o->cov || !o->triplets || o->capacity < 1)
    return fail(h, CKF_E_ARG, "null output array");
  const int nb = h->geo.n_barrel;
  if (sc->layer_b < 0 || sc->layer_t >= nb || !(sc->layer_b < sc->layer_m && sc->layer_m < sc->layer_t))
    return fail(h, CKF_E_ARG, "seeding layers must be barrel layers with bottom < middle < top");
  if (!(sc->dphi_max > 0.0 && sc->dphi_max < 1.5) || !(sc->cot_max > 0.0) || !(sc->pt_min > 0.0))
    return fail(h, CKF_E_ARG, "bad seeding cuts");
  cudaStream_t st = (cudaStream_t)stream;
  std::lock_guard<std::mutex> lk(h->mu);
  cudaStreamWaitEvent(st, h->seed_done, 0);   // one workspace: calls are ordered one after the other
  const int rc = h->cfg.precision == 32 ? launch_seed<float>(h, m, sc, o, st) : launch_seed<double>(h, m, sc, o, st);
  cudaEventRecord(h->seed_done, st);
  return rc;
}

int ckf_resolve(ckf_handle* h, const ckf_tracks* t, int32_t n_measurements, ckf_resolution* o, void* stream) {
  if (!h) return CKF_E_ARG;
  if (!t || !o) return fail(h, CKF_E_ARG, "null argument");
  if (!t->n_tracks || !t->track_offsets || !t->meas_idx || !t->chi2_sum) return fail(h, CKF_E_ARG, "null input array");
  if (!o->accepted || !o->n_shared || !o->summary) return fail(h, CKF_E_ARG, "null output array");
  if (n_measurements < 0 || n_measurements > h->cfg.max_measurements)
    return fail(h, CKF_E_CAPACITY, "n_measurements %d exceeds capacity %d", n_measurements, h->cfg.max_measurements);
  if (h->cfg.max_tracks > (1 << 24)) return fail(h, CKF_E_CAPACITY, "ckf_resolve ranks at most 2^24 candidates");
  if (o->max_shared_hits < 0 || !(o->max_shared_fraction >= 0.0)) return fail(h, CKF_E_ARG, "bad sharing limits");
  cudaStream_t st = (cudaStream_t)stream;
  std::lock_guard<std::mutex> lk(h->mu);
  cudaStreamWaitEvent(st, h->resolve_done, 0);   // one workspace: resolutions are ordered one after the other
  cudaError_t e;
  if (h->cfg.precision == 32) {
    ResolveParams<float> p{t->n_tracks, t->track_offsets, t->meas_idx, (const float*)t->chi2_sum, h->cfg.max_tracks,
                           n_measurements, o->max_shared_hits, o->max_shared_fraction, h->rs_key, h->rs_best, h->rs_owner,
                           h->rs_state, h->rs_g, o->accepted, o->n_shared, o->summary};
    void* args[] = {&p};
    e = cudaLaunchCooperativeKernel((void*)ckf_resolve_kernel<float>, dim3(h->resolve_grid), dim3(RESOLVE_NT), args, 0, st);
  } else {
    ResolveParams<double> p{t->n_tracks, t->track_offsets, t->meas_idx, (const double*)t->chi2_sum, h->cfg.max_tracks,
                            n_measurements, o->max_shared_hits, o->max_shared_fraction, h->rs_key, h->rs_best, h->rs_owner,
                            h->rs_state, h->rs_g, o->accepted, o->n_shared, o->summary};
    void* args[] = {&p};
    e = cudaLaunchCooperativeKernel((void*)ckf_resolve_kernel<double>, dim3(h->resolve_grid), dim3(RESOLVE_NT), args, 0, st);
  }
  cudaEventRecord(h->resolve_done, st);
  if (e != cudaSuccess) return fail(h, CKF_E_CUDA, "ckf_resolve launch failed: %s", cudaGetErrorString(e));
  return CKF_OK;
}

// ckf_resolve without a handle and without allocation: scratch in g_resolve_static_scratch (see include/ckf.h).
int ckf_resolve_static(const ckf_tracks* t, int32_t max_tracks, int32_t n_measurements, int32_t precision,
                       ckf_resolution* o, void* stream) {
  ckf_handle* h = nullptr;  // for fail() / CK(): the message goes to the calling thread's slot
  if (!t || !o) return fail(h, CKF_E_ARG, "ckf_resolve_static: null argument");
  if (!t->n_tracks || !t->track_offsets || !t->meas_idx || !t->chi2_sum) return fail(h, CKF_E_ARG, "ckf_resolve_static: null input array");
  if (!o->accepted || !o->n_shared || !o->summary) return fail(h, CKF_E_ARG, "ckf_resolve_static: null output array");
  if (precision != 32 && precision != 64) return fail(h, CKF_E_ARG, "ckf_resolve_static: precision must be 32 or 64");
  if (o->max_shared_hits < 0 || !(o->max_shared_fraction >= 0.0)) return fail(h, CKF_E_ARG, "ckf_resolve_static: bad sharing limits");
  if (max_tracks < 1 || max_tracks > CKF_RESOLVE_STATIC_MAX_TRACKS)
    return fail(h, CKF_E_CAPACITY, "ckf_resolve_static: max_tracks %d outside 1..%d (the static scratch array is sized for that; use ckf_resolve)",
                max_tracks, CKF_RESOLVE_STATIC_MAX_TRACKS);
  if (n_measurements < 0 || n_measurements > CKF_RESOLVE_STATIC_MAX_MEASUREMENTS)
    return fail(h, CKF_E_CAPACITY, "ckf_resolve_static: n_measurements %d outside 0..%d (the static scratch array is sized for that; use ckf_resolve)",
                n_measurements, CKF_RESOLVE_STATIC_MAX_MEASUREMENTS);
  // set-up, once per device, with that device current: address of the array, and the grid a cooperative launch may have
  struct PerDevice { unsigned char* base = nullptr; int grid32 = 0, grid64 = 0; bool ready = false; };
  static PerDevice s_dev[64];
  static std::mutex s_mu;
  int dev = -1;
  CK(cudaGetDevice(&dev));
  if (dev < 0 || dev >= 64) return fail(h, CKF_E_ARG, "ckf_resolve_static: device ordinal %d not supported", dev);
  PerDevice pd;
  {
    std::lock_guard<std::mutex> lk(s_mu);
    if (!s_dev[dev].ready) {
      void* ptr = nullptr;
      CK(cudaGetSymbolAddress(&ptr, g_resolve_static_scratch));
      int sms = 0, b32 = 0, b64 = 0;
      CK(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
      CK(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&b32, ckf_resolve_kernel<float>, RESOLVE_NT, 0));
      CK(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&b64, ckf_resolve_kernel<double>, RESOLVE_NT, 0));
      s_dev[dev].base = (unsigned char*)ptr;
      s_dev[dev].grid32 = std::max(1, b32) * sms;   // a cooperative launch needs every block resident
      s_dev[dev].grid64 = std::max(1, b64) * sms;
      s_dev[dev].ready = true;
    }
    pd = s_dev[dev];
  }
  constexpr size_t MT = CKF_RESOLVE_STATIC_MAX_TRACKS, MM = CKF_RESOLVE_STATIC_MAX_MEASUREMENTS;
  unsigned long long* key = (unsigned long long*)pd.base;                       // [MT]
  unsigned long long* best = (unsigned long long*)(pd.base + MT * 8);           // [2][n_measurements], room for [2][MM]
  int32_t* owner = (int32_t*)(pd.base + MT * 8 + MM * 16);                      // [MM]
  int32_t* state = (int32_t*)(pd.base + MT * 8 + MM * 20);                      // [MT]
  int32_t* g = (int32_t*)(pd.base + MT * 12 + MM * 20);                         // [4]
  static_assert(MT * 12 + MM * 20 + 16 <= CKF_RESOLVE_STATIC_SCRATCH_BYTES, "scratch layout");
  // the kernel initialises keys, minima, owners, states and counters for the sizes of THIS call before it reads them
  // (the array keeps the previous call's contents)
  cudaStream_t st = (cudaStream_t)stream;
  cudaError_t e;
  if (precision == 32) {
    ResolveParams<float> p{t->n_tracks, t->track_offsets, t->meas_idx, (const float*)t->chi2_sum, max_tracks, n_measurements,
                           o->max_shared_hits, o->max_shared_fraction, key, best, owner, state, g, o->accepted, o->n_shared,
                           o->summary};
    void* args[] = {&p};
    e = cudaLaunchCooperativeKernel((void*)ckf_resolve_kernel<float>, dim3(pd.grid32), dim3(RESOLVE_NT), args, 0, st);
  } else {
    ResolveParams<double> p{t->n_tracks, t->track_offsets, t->meas_idx, (const double*)t->chi2_sum, max_tracks, n_measurements,
                            o->max_shared_hits, o->max_shared_fraction, key, best, owner, state, g, o->accepted, o->n_shared,
                            o->summary};
    void* args[] = {&p};
    e = cudaLaunchCooperativeKernel((void*)ckf_resolve_kernel<double>, dim3(pd.grid64), dim3(RESOLVE_NT), args, 0, st);
  }
  if (e != cudaSuccess) return fail(h, CKF_E_CUDA, "ckf_resolve_static launch failed: %s", cudaGetErrorString(e));
  return CKF_OK;
}

int ckf_get_counters(ckf_handle* h, void* stream, ckf_counters* out) {
  if (!h || !out) return CKF_E_ARG;
  cudaStream_t st = (cudaStream_t)stream;
  Workspace* w = nullptr;
  {
    std::lock_guard<std::mutex> lk(h->mu);
    for (auto& x : h->ws)
      if (x.used && x.stream_tag == (void*)st) { w = &x; break; }
  }
  if (!w) return fail(h, CKF_E_ARG, "no ckf_find was issued on this stream");
  unsigned long long c[CNT_N];
  CK(cudaStreamSynchronize(st));
  CK(cudaMemcpy(c, w->counters, sizeof(c), cudaMemcpyDeviceToHost));
  out->tips = (int64_t)c[CNT_TIPS]; out->visits = (int64_t)c[CNT_VISITS]; out->rk_trials = (int64_t)c[CNT_TRIALS];
  out->rk_accepted = (int64_t)c[CNT_ACCEPTED]; out->gate_tests = (int64_t)c[CNT_GATE];
  out->updates = (int64_t)c[CNT_UPDATES]; out->links = (int64_t)c[CNT_LINKS]; out->iterations = (int64_t)c[CNT_ITER];
  out->gate_tests_executed = (int64_t)c[CNT_GATE_EXEC];
  return CKF_OK;
}

int ckf_set_timing(ckf_handle* h, int on) {
  if (!h) return CKF_E_ARG;
  h->timing = on != 0 || h->timing_print;
  return CKF_OK;
}

int ckf_get_timing(ckf_handle* h, void* stream, ckf_timing* out) {
  if (!h || !out) return CKF_E_ARG;
  cudaStream_t st = (cudaStream_t)stream;
  Workspace* w = nullptr;
  {
    std::lock_guard<std::mutex> lk(h->mu);
    for (auto& x : h->ws)
      if (x.used && x.stream_tag == (void*)st) { w = &x; break; }
  }
  if (!w) return fail(h, CKF_E_ARG, "no ckf_find was issued on this stream");
  out->init_ms = w->last_ms[0]; out->sort_ms = w->last_ms[1]; out->step_ms = w->last_ms[2]; out->visit_ms = w->last_ms[3];
  out->scan_ms = w->last_ms[5]; out->update_ms = w->last_ms[6];
  out->emit_ms = w->last_ms[7] + w->last_ms[8] + w->last_ms[9];
  out->launches = w->last_launches;
  return CKF_OK;
}

int ckf_get_launch_info(const ckf_handle* h, int32_t* blocks, int32_t* threads, int32_t* smem, int32_t* regs) {
  if (!h) return CKF_E_ARG;
  if (blocks) *blocks = h->step_grid;
  if (threads) *threads = STEP_NT;
  if (smem) *smem = (int32_t)((STEP_NT / 32) * PickSmem::bytes());
  if (regs) *regs = h->step_regs;
  return CKF_OK;
}

// Measured plain-ALU peak (see ckf_peak.cuh).  mix: 0 = float32 FMA chains only, 1 = float64 only, 2 = both at once
// (8 float + 4 double chains per thread: the two pipes fed together).  Launches back to back for at least `seconds`
// on the default stream; *tflops_f32 / *tflops_f64 receive the flop rates over the whole run (an FMA = 2 flop),
// *best_* the rates of the fastest single launch.
int ckf_measure_alu_peak(int mix, double seconds, double* tflops_f32, double* tflops_f64, double* best_f32, double* best_f64) {
  ckf_handle* h = nullptr;
  if (mix < 0 || mix > 2 || !(seconds > 0.0) || !tflops_f32 || !tflops_f64) return fail(h, CKF_E_ARG, "bad argument");
  int dev = 0, sms = 0;
  CK(cudaGetDevice(&dev));
  CK(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
  const int blocks = sms * 8, threads = 256, iters = 4096;
  double* out = nullptr;
  CK(cudaMalloc(&out, (size_t)blocks * threads * sizeof(double)));
  const int nf = mix == 0 ? 8 : (mix == 2 ? 8 : 0), nd = mix == 1 ? 8 : (mix == 2 ? 4 : 0);
  auto launch = [&]() {
    if (mix == 0) ckf_fma_chain<8, 0><<<blocks, threads>>>(out, iters, 0.999f, 1e-3f, 0.999, 1e-3);
    else if (mix == 1) ckf_fma_chain<0, 8><<<blocks, threads>>>(out, iters, 0.999f, 1e-3f, 0.999, 1e-3);
    else ckf_fma_chain<8, 4><<<blocks, threads>>>(out, iters, 0.999f, 1e-3f, 0.999, 1e-3);
  };
  cudaEvent_t e0, e1, a, b;
  cudaEventCreate(&e0); cudaEventCreate(&e1); cudaEventCreate(&a); cudaEventCreate(&b);
  for (int i = 0; i < 3; ++i) launch();
  cudaDeviceSynchronize();
  const double per_launch = (double)blocks * threads * (double)iters * 8.0 * 2.0;   // flop per chain kind per chain
  double total_ms = 0.0, best_ms = 1e30;
  long n = 0;
  cudaEventRecord(e0);
  while (total_ms < seconds * 1e3) {
    cudaEventRecord(a);
    for (int i = 0; i < 8; ++i) launch();
    cudaEventRecord(b);
    cudaEventSynchronize(b);
    float ms = 0.f;
    cudaEventElapsedTime(&ms, a, b);
    best_ms = ms / 8.0 < best_ms ? ms / 8.0 : best_ms;
    n += 8;
    cudaEventRecord(e1);
    cudaEventSynchronize(e1);
    cudaEventElapsedTime(&ms, e0, e1);
    total_ms = ms;
  }
  cudaError_t e = cudaGetLastError();
  cudaEventDestroy(e0); cudaEventDestroy(e1); cudaEventDestroy(a); cudaEventDestroy(b);
  cudaFree(out);
  if (e != cudaSuccess) return fail(h, CKF_E_CUDA, "fma chain failed: %s", cudaGetErrorString(e));
  *tflops_f32 = nf * per_launch * (double)n / (total_ms * 1e-3) / 1e12;
  *tflops_f64 = nd * per_launch * (double)n / (total_ms * 1e-3) / 1e12;
  if (best_f32) *best_f32 = nf * per_launch / (best_ms * 1e-3) / 1e12;
  if (best_f64) *best_f64 = nd * per_launch / (best_ms * 1e-3) / 1e12;
  return CKF_OK;
}

int ckf_destroy(ckf_handle* h) {
  if (!h) return CKF_E_ARG;
  cudaDeviceSynchronize();
  for (auto& w : h->ws) {
    if (w.graph_exec) cudaGraphExecDestroy(w.graph_exec);
    if (w.cap_stream) cudaStreamDestroy(w.cap_stream);
    if (w.done) cudaEventDestroy(w.done);
    if (w.pinned_nt) cudaFreeHost(w.pinned_nt);
  }
  if (h->fit_done) cudaEventDestroy(h->fit_done);
  if (h->resolve_done) cudaEventDestroy(h->resolve_done);
  if (h->seed_done) cudaEventDestroy(h->seed_done);
  for (void* p : h->allocs) cudaFree(p);
  delete h;
  return CKF_OK;
}

}  // extern "C"
