// C ABI of the pasta library (include/pasta.h): argument validation, buffer ownership and the order in
// which the kernels of one MD step are enqueued.  No arithmetic of the method lives here except the
// host-side bookkeeping of the box length (L_{k+1} = s L_k in FP64, reading D9).
#include <math.h>
#include <stdarg.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <new>

#include "pasta_internal.cuh"

namespace pasta {

static thread_local char g_error[512] = "";

void set_error(const char* fmt, ...) {
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(g_error, sizeof(g_error), fmt, ap);
  va_end(ap);
}

int buffer_reserve(Sim* s, Buffer* b, size_t bytes) {
  if (bytes <= b->bytes && b->ptr) return PASTA_OK;
  buffer_release(s, b);
  // grow geometrically so that an expanding box does not reallocate every few steps
  size_t want = bytes + bytes / 4 + 256;
  void* p = nullptr;
  if (s->env.alloc) {
    p = s->env.alloc(want, s->env.user);
  } else {
    if (cudaMalloc(&p, want) != cudaSuccess) p = nullptr;
  }
  if (!p) {
    set_error("device allocation of %zu bytes failed", want);
    return PASTA_ENOMEM;
  }
  b->ptr = p;
  b->bytes = want;
  s->state_gen += 1;  // a captured step holds the old pointer
  return PASTA_OK;
}

void buffer_release(Sim* s, Buffer* b) {
  if (!b->ptr) return;
  // pending work on the stream may still use the buffer.  While a step is being captured s->stream is the capture
  // stream: synchronising it is illegal (it would invalidate the capture) and it carries no pending work anyway --
  // the kernels of the previous steps are on the caller's stream.  (A buffer that moves bumps state_gen, so the
  // capture under way is discarded and the step redone kernel by kernel.)
  cudaStreamSynchronize(s->graph.capturing ? s->graph.home : s->stream);
  if (s->env.alloc && s->env.free)
    s->env.free(b->ptr, s->env.user);
  else if (!s->env.alloc)
    cudaFree(b->ptr);
  b->ptr = nullptr;
  b->bytes = 0;
}

static void release_all(Sim* s) {
  s->e = Buffer();  // an alias into s->F's allocation (pasta_create), nothing of its own to free
  Buffer* bs[] = {&s->x, &s->v, &s->F, &s->is_p, &s->cell_id, &s->bin_count, &s->bin_start, &s->scan_tmp,
                  &s->perm, &s->perm_raw, &s->pos4, &s->cxyz, &s->cpos, &s->partials, &s->scalars, &s->counters, &s->cl_parent, &s->cl_A,
                  &s->cl_Z, &s->cl_cell_id, &s->cl_count, &s->cl_start, &s->cl_perm, &s->chunk_tab, &s->chunk_first, &s->xref, &s->slot_of, &s->list_off,
                  &s->list_pool};
  for (Buffer* b : bs) buffer_release(s, b);
}

static int check_sim(const Sim* s) {
  if (!s) {
    set_error("pasta_sim handle is NULL");
    return PASTA_EINVAL;
  }
  return PASTA_OK;
}

static int use_device(const Sim* s) {
  PASTA_CUDA_OK(cudaSetDevice(s->env.device));
  return PASTA_OK;
}

static void timing_collect(Sim* s) {
  for (size_t k = 0; k < s->ev_kind.size(); ++k) {
    float ms = 0.f;
    cudaEventSynchronize(s->evs[2 * k + 1]);
    if (cudaEventElapsedTime(&ms, s->evs[2 * k], s->evs[2 * k + 1]) == cudaSuccess) s->ms_acc[s->ev_kind[k]] += ms;
  }
  s->ev_kind.clear();
  s->ev_used = 0;
}

// Brackets a kernel group with a fresh pair of events (drained lazily, so timing does not serialise
// the host against the stream more often than once per 1024 groups).
struct Timer {
  Sim* s;
  bool on;
  Timer(Sim* s_, int which) : s(s_), on(s_->timing) {
    if (!on) return;
    if (s->ev_used >= 2048) timing_collect(s);
    while (s->evs.size() < s->ev_used + 2) {
      cudaEvent_t e = nullptr;
      cudaEventCreate(&e);
      s->evs.push_back(e);
    }
    s->ev_kind.push_back(which);
    cudaEventRecord(s->evs[s->ev_used], s->stream);
  }
  ~Timer() {
    if (!on) return;
    cudaEventRecord(s->evs[s->ev_used + 1], s->stream);
    s->ev_used += 2;
  }
};

// One force evaluation of the current positions.  Dense regime: sort + chunk table (K1), chunk kernel (K2).  Where
// list_mode_wanted(): the paper's neighbour list -- sort, chunk table and per-chunk source lists are
// built with a halo and reused; every evaluation first refreshes the sorted coordinates and reads back the largest
// displacement D since the build, and rebuilds when a pair could have entered the reach unseen:
//   own + source displacement 2 D > halo  (less reach (L0/L - 1) if the box has shrunk since).
// The sorted slots whose targets this rank evaluates (pasta_set_shard): the whole range on one GPU.
static int shard_window(Sim* s) {
  s->shard.slot_lo = 0;
  s->shard.slot_hi = 0x7fffffff;
  if (s->shard.world <= 1) return PASTA_OK;
  std::vector<int64_t> b((size_t)s->shard.world + 1);
  double cost[2];
  PASTA_TRY(pasta_shard_costs(reinterpret_cast<const pasta_sim*>(s), cost));
  PASTA_TRY(pasta_shard_bounds(s->N, s->Np, cost[0], cost[1], s->shard.world, b.data()));
  s->shard.slot_lo = (int32_t)b[(size_t)s->shard.rank];
  s->shard.slot_hi = (int32_t)b[(size_t)s->shard.rank + 1];
  return PASTA_OK;
}

static int evaluate_forces_tail(Sim* s, bool with_energy, double kick = 0.0) {
  s->n_force_evals += 1;
  const bool sharded = s->shard.world > 1;
  PASTA_TRY(shard_window(s));
  {
    Timer t(s, 1);
    // the other ranks' targets stay zero: the sum over ranks then completes every particle exactly.  F and e are one
    // contiguous run ([F | e], pasta_create): one memset and one collective cover both
    const size_t shard_doubles = (with_energy ? 4 : 3) * (size_t)s->N;
    if (sharded) PASTA_CUDA_OK(cudaMemsetAsync(s->F.ptr, 0, 8 * shard_doubles, s->stream));
    if (s->list.valid) PASTA_TRY(k2_list_forces(s, with_energy));
    else PASTA_TRY(k2_forces(s, with_energy, kick));
    if (s->prm.coulomb_all_pairs) PASTA_TRY(k2_coulomb_all_pairs(s, with_energy));
    if (sharded) {
      if (s->shard.allreduce(s->F.ptr, (int64_t)shard_doubles, s->shard.user) != 0) {
        set_error("pasta_set_shard: the allreduce callback failed");
        return PASTA_ECUDA;
      }
    }
  }
  if (s->timing) s->n_timed += 1;
  s->forces_valid = true;
  s->energies_valid = with_energy;
  return PASTA_OK;
}

// kick != 0 (a caller that has checked kick_can_ride): the chunk kernel adds v += kick F as it writes F.
static bool kick_can_ride(const Sim* s) {
  return s->tune.force_variant == 0 && s->shard.world <= 1 && !s->prm.coulomb_all_pairs && !s->list.valid && !list_mode_wanted(s);
}
static int evaluate_forces(Sim* s, bool with_energy, double kick = 0.0) {
  {
    Timer t(s, 0);
    if (s->list.valid) {
      double d = 0.0;
      if (s->list.pending) PASTA_TRY(k1_refresh_wait(s, &d));  // the kick-drift kernel of this step carried the refresh
      else PASTA_TRY(k1_refresh(s, &d));
      const double ratio = s->L / s->list.L0;
      const double delta = s->list.halo + (ratio >= 1.0 ? 0.0 : s->prm.r_c * (1.0 - 1.0 / ratio));
      // (the frozen grid scales with the box: 5 % keeps the cells within the width the FP32 coordinates are good for)
      if (!(2.0 * d <= delta) || ratio > 1.05 || ratio < 0.95 || !list_mode_wanted(s)) s->list.valid = false;
    }
    if (!s->list.valid) {
      const bool lists = list_mode_wanted(s);
      PASTA_TRY(k1_build(s));
      s->n_list_builds += 1;
      if (lists) {
        const double halo = list_halo(s);
        const int rc = k2_list_build(s, halo);
        if (rc == 1) {  // too dense for lists after all (a clustered state): the chunk kernel on its own sort, until the
          s->no_lists = true;  // caller brings another state or box (pasta_set_state*, pasta_expand try lists again)
          PASTA_TRY(k1_build(s));
          return evaluate_forces_tail(s, with_energy);
        }
        PASTA_TRY(rc);
        PASTA_TRY(buffer_reserve(s, &s->xref, 24 * (size_t)s->N));
        PASTA_CUDA_OK(cudaMemcpyAsync(s->xref.ptr, s->x.ptr, 24 * (size_t)s->N, cudaMemcpyDeviceToDevice, s->stream));
        s->list.L0 = s->L;
        s->list.halo = halo;
        s->list.valid = true;
      }
    }
  }
  return evaluate_forces_tail(s, with_energy, kick);
}

// A step on reused neighbour lists without a round trip to the host in its critical path: the
// kick-drift kernel refreshes the frozen order, measures the largest displacement since the build and DECIDES on the
// device whether the lists survive (2 D <= halo); the force kernel -- with the second half kick riding along -- is
// enqueued right behind it and returns at once if they do not.  The host reads the same decision from its mailbox
// while the force kernel runs; only when the trigger has fired does it rebuild and evaluate again.
static int list_step(Sim* s, double dt, double sc, double L_wrap, bool energy, bool rescale, bool* done) {
  *done = false;
  const double ratio = s->L / s->list.L0;
  // what the host alone can tell: the frozen grid is still good for this box, and lists are still wanted in it
  if (ratio > 1.05 || ratio < 0.95 || !list_mode_wanted(s) || s->shard.world > 1 || s->prm.coulomb_all_pairs) return PASTA_OK;
  {
    Timer t(s, 2);
    PASTA_TRY(k3_kick_drift_refresh(s, dt, sc, L_wrap));
    s->lin_n += 1;
  }
  s->clusters_valid = false;
  *done = true;
  const double h2 = dt / (2.0 * s->prm.mass);
  {
    Timer t(s, 1);
    PASTA_TRY(k2_list_forces(s, energy, true, rescale ? 0.0 : h2));
  }
  double d = 0.0;
  PASTA_TRY(k1_refresh_wait(s, &d));
  const double delta = s->list.halo + (ratio >= 1.0 ? 0.0 : s->prm.r_c * (1.0 - 1.0 / ratio));
  if (2.0 * d <= delta) {  // (the device took the same decision in the same arithmetic)
    s->n_force_evals += 1;
    if (s->timing) s->n_timed += 1;
    s->forces_valid = true;
    s->energies_valid = energy;
    s->step_count += 1;
    if (rescale) {
      Timer t(s, 2);
      PASTA_TRY(k3_kick_ke(s, dt, true));
    }
    return PASTA_OK;
  }
  // the gated kernel did nothing: rebuild, evaluate, kick
  s->list.valid = false;
  s->forces_valid = false;
  PASTA_TRY(evaluate_forces(s, energy));
  s->step_count += 1;
  {
    Timer t(s, 2);
    PASTA_TRY(k3_kick_ke(s, dt, rescale));
  }
  return PASTA_OK;
}

// One MD step with s->L already set to the box the forces are evaluated in (O2: first half kick + drift, forces,
// second half kick, rescale on every thermostat_interval-th step).
static int step_body(Sim* s, double dt, double sc, double L_wrap, bool energy, bool rescale) {
  if (s->list.valid) {
    bool done = false;
    PASTA_TRY(list_step(s, dt, sc, L_wrap, energy, rescale, &done));
    if (done) return PASTA_OK;
  }
  {
    Timer t(s, 2);
    // the cell histogram of the new positions rides along unless the sorted order is frozen (or about to be
    // rebuilt on the lists' own grid)
    if (s->list.valid) PASTA_TRY(k3_kick_drift_refresh(s, dt, sc, L_wrap));
    else PASTA_TRY(k3_kick_drift_count(s, dt, sc, L_wrap, !list_mode_wanted(s)));
    s->lin_n += 1;
  }
  s->clusters_valid = false;
  // a plain step on the chunk path: the second half kick rides along with the force write of the pair kernel; a step
  // that ends with the rescale needs the kinetic energy and keeps the kick kernel
  const bool ride = !rescale && kick_can_ride(s);
  PASTA_TRY(evaluate_forces(s, energy, ride ? dt / (2.0 * s->prm.mass) : 0.0));
  s->step_count += 1;
  if (!ride) {
    Timer t(s, 2);
    PASTA_TRY(k3_kick_ke(s, dt, rescale));
  }
  return PASTA_OK;
}

static void graphs_drop(Sim* s) {
  for (int w = 0; w < 2; ++w) {
    if (s->graph.exec[w]) cudaGraphExecDestroy(s->graph.exec[w]);
    s->graph.exec[w] = nullptr;
  }
  s->graph.gen = -1;
  s->graph.warm = 0;
}
static void graphs_destroy(Sim* s) {
  graphs_drop(s);
  if (s->graph.cap) cudaStreamDestroy(s->graph.cap);
  s->graph.cap = nullptr;
}

// A fixed-box step on the chunk path enqueues the same 8-10 kernels with the same arguments every time (SURVEY 3b:
// "capture the step in a CUDA graph"): after two such steps have run kernel by kernel (every buffer has its final size
// by then) the step is captured once per kind (plain / ending with the rescale) and replayed with one launch.
// Anything that changes a captured argument -- a buffer that moved, a new particle set, another dt or box -- drops
// the graphs; timing brackets, a scaling box and the neighbour-list regime always take the kernel-by-kernel path.
static int step_once(Sim* s, double dt, double sc, double L_wrap, bool energy, bool rescale) {
  const bool eligible = s->tune.graphs != 0 && sc == 1.0 && !(s->prm.xi_dot > 0.0) && !s->timing && !s->list.valid &&
                        s->tune.force_variant == 0 && s->forces_valid && !list_mode_wanted(s) && s->sort_kind == 0 &&
                        s->shard.world <= 1 &&
                        s->bins_zeroed >= s->grid_sp[0].nc3 + s->grid_sp[1].nc3 + 1;
  if (!eligible) {
    s->graph.warm = 0;
    return step_body(s, dt, sc, L_wrap, energy, rescale);
  }
  if (s->graph.gen != s->state_gen || s->graph.L != s->L || s->graph.dt != dt || s->graph.energy != (int)energy) {
    graphs_drop(s);
    s->graph.gen = s->state_gen;
    s->graph.L = s->L;
    s->graph.dt = dt;
    s->graph.energy = (int)energy;
  }
  const int w = rescale ? 1 : 0;
  if (!s->graph.exec[w]) {
    if (s->graph.warm < 2) {
      s->graph.warm += 1;
      const int rc = step_body(s, dt, sc, L_wrap, energy, rescale);
      if (s->graph.gen != s->state_gen) s->graph.warm = 0;  // a buffer grew during this step: not settled yet
      return rc;
    }
    // capture this step; the host-side bookkeeping of step_body runs now, its kernels when the graph is launched
    const int64_t launches0 = s->launches;
    if (!s->graph.cap && cudaStreamCreateWithFlags(&s->graph.cap, cudaStreamNonBlocking) != cudaSuccess) s->graph.cap = nullptr;
    if (!s->graph.cap || cudaStreamBeginCapture(s->graph.cap, cudaStreamCaptureModeThreadLocal) != cudaSuccess) {
      cudaGetLastError();
      s->tune.graphs = 0;
      return step_body(s, dt, sc, L_wrap, energy, rescale);
    }
    cudaStream_t const user_stream = s->stream;
    s->graph.home = user_stream;
    s->graph.capturing = true;
    s->stream = s->graph.cap;
    const int rc = step_body(s, dt, sc, L_wrap, energy, rescale);
    s->stream = user_stream;
    s->graph.capturing = false;
    cudaGraph_t g = nullptr;
    const cudaError_t ce = cudaStreamEndCapture(s->graph.cap, &g);
    if (rc != PASTA_OK || ce != cudaSuccess || !g || s->graph.gen != s->state_gen) {
      if (g) cudaGraphDestroy(g);
      cudaGetLastError();
      s->tune.graphs = 0;
      s->forces_valid = false;  // the captured kernels never ran: positions, velocities and forces are those of the
      s->hist_valid = false;    // step before; undo the bookkeeping and redo the step kernel by kernel
      s->bins_zeroed = 0;
      s->step_count -= 1;
      s->lin_n -= 1;
      s->n_force_evals -= 1;
      s->n_list_builds -= 1;
      s->launches = launches0;
      if (rc != PASTA_OK) return rc;
      PASTA_TRY(evaluate_forces(s, energy));
      return step_body(s, dt, sc, L_wrap, energy, rescale);
    }
    const cudaError_t ie = cudaGraphInstantiate(&s->graph.exec[w], g, 0);
    cudaGraphDestroy(g);
    if (ie != cudaSuccess) {
      set_error("cudaGraphInstantiate failed: %s", cudaGetErrorString(ie));
      return PASTA_ECUDA;
    }
    s->graph.launches[w] = s->launches - launches0;
    PASTA_CUDA_OK(cudaGraphLaunch(s->graph.exec[w], s->stream));
    s->graph.replays += 1;
    return PASTA_OK;
  }
  // replay: the bookkeeping of step_body, then one launch
  PASTA_CUDA_OK(cudaGraphLaunch(s->graph.exec[w], s->stream));
  s->lin_n += 1;
  s->step_count += 1;
  s->clusters_valid = false;
  s->n_force_evals += 1;
  s->n_list_builds += 1;
  s->hist_valid = false;
  s->forces_valid = true;
  s->energies_valid = energy;
  s->launches += s->graph.launches[w];
  s->graph.replays += 1;
  return PASTA_OK;
}

}  // namespace pasta

using namespace pasta;

extern "C" {

const char* pasta_last_error(void) { return g_error; }
const char* pasta_version(void) { return "pasta-b200 0.1 (sm_100a)"; }

int pasta_params_default(pasta_params* p) {
  if (!p) {
    set_error("params pointer is NULL");
    return PASTA_EINVAL;
  }
  memset(p, 0, sizeof(*p));
  p->struct_size = (uint32_t)sizeof(pasta_params);
  p->a = 110.0;
  p->b = -26.0;
  p->c = 24.0;
  p->Lambda = 1.25;
  p->alpha_hbarc = 1.44;
  p->lambda = 10.0;
  p->r_c = 20.0;
  p->mass = 939.0;
  p->scale_per_step = 1.0;
  p->thermostat_interval = 0;
  p->cell_subdiv = 4;
  p->energy_every_step = 1;
  p->skip_exact_zeros = 1;
  p->list_reuse = 1;
  p->list_halo = 0.0;
  p->r_nuc = 0.0;
  p->xi_dot = 0.0;
  p->coulomb_all_pairs = 0;
  return PASTA_OK;
}

// Smallest box side a parameter set may run in: 2 r_c (one nearest image within the cut-off; D3) and, with
// coulomb_all_pairs, PASTA_COULOMB_ALL_PAIRS_MIN_L (pasta.h; D26).
static double min_box_side(const pasta_params& p) {
  const double two_rc = 2.0 * p.r_c;
  return p.coulomb_all_pairs != 0 && two_rc < PASTA_COULOMB_ALL_PAIRS_MIN_L ? PASTA_COULOMB_ALL_PAIRS_MIN_L : two_rc;
}
static int check_box_side(const pasta_params& p, double L, const char* who) {
  if (L > 0.0 && p.r_c <= 0.5 * L && L >= min_box_side(p)) return PASTA_OK;
  if (L > 0.0 && p.r_c <= 0.5 * L)
    set_error("%s: coulomb_all_pairs needs a box side of at least %g fm (got %g): the nearest image of a proton pair is "
              "decided in FP32 box fractions, and the force error of a pair that lands on the wrong side of L/2 is "
              "only negligible from there on (pasta.h)", who, (double)PASTA_COULOMB_ALL_PAIRS_MIN_L, L);
  else
    set_error("%s: need L >= 2 r_c (L = %g, r_c = %g): the nearest image would be ambiguous", who, L, p.r_c);
  return PASTA_EINVAL;
}

static int validate_params(const pasta_params* p, double L) {
  if (!p || p->struct_size != sizeof(pasta_params)) {
    set_error("pasta_params is NULL or has the wrong struct_size");
    return PASTA_EINVAL;
  }
  if (!(p->r_c > 0) || !(p->Lambda > 0) || !(p->lambda > 0) || !(p->mass > 0) || !(p->scale_per_step > 0) ||
      p->thermostat_interval < 0 || p->cell_subdiv < 1 || p->cell_subdiv > 64 || !(p->list_halo >= 0.0)) {
    set_error("pasta_params: r_c, Lambda, lambda, mass, scale_per_step must be > 0, thermostat_interval >= 0, "
              "1 <= cell_subdiv <= 64, list_halo >= 0");
    return PASTA_EINVAL;
  }
  if (!(p->r_nuc >= 0.0) || p->r_nuc > p->r_c) {
    set_error("pasta_params: need 0 <= r_nuc <= r_c");
    return PASTA_EINVAL;
  }
  if (p->coulomb_all_pairs != 0 && !(p->r_nuc > 0.0)) {
    set_error("pasta_params: coulomb_all_pairs needs r_nuc > 0 (without a Coulomb cut-off r_nuc is what cuts the nuclear terms)");
    return PASTA_EINVAL;
  }
  if (!(p->xi_dot >= 0.0) || (p->xi_dot > 0.0 && p->scale_per_step != 1.0)) {
    set_error("pasta_params: need xi_dot >= 0, and scale_per_step == 1 when xi_dot > 0");
    return PASTA_EINVAL;
  }
  if (p->r_c > 0.5 * L) {
    set_error("r_c = %g exceeds L/2 = %g: the nearest image would be ambiguous", p->r_c, 0.5 * L);
    return PASTA_EINVAL;
  }
  return check_box_side(*p, L, "pasta_create");
}

int pasta_create(pasta_sim** out, int64_t N, double Y_P, double density, double T, const pasta_params* p,
                 uint64_t seed, const pasta_env* env) {
  if (!out) {
    set_error("out is NULL");
    return PASTA_EINVAL;
  }
  *out = nullptr;
  if (N <= 0 || N >= (1ll << 26) || !(Y_P >= 0.0 && Y_P <= 1.0) || !(density > 0.0) || !(T >= 0.0)) {
    set_error("pasta_create: need 0 < N < 2^26, 0 <= Y_P <= 1, density > 0, T >= 0");
    return PASTA_EINVAL;
  }
  const double L = cbrt((double)N / density);
  PASTA_TRY(validate_params(p, L));
  if (env && env->struct_size != sizeof(pasta_env)) {
    set_error("pasta_env has the wrong struct_size");
    return PASTA_EINVAL;
  }
  Sim* s = new (std::nothrow) Sim();
  if (!s) {
    set_error("host allocation failed");
    return PASTA_ENOMEM;
  }
  s->prm = *p;
  {
    auto env_int = [](const char* name, int dflt) {
      const char* v = getenv(name);
      return v && *v ? atoi(v) : dflt;
    };
    s->tune.force_variant = env_int("PASTA_FORCE_VARIANT", 0);
    s->tune.auto_grid = env_int("PASTA_AUTO_GRID", 1);
    s->tune.x_subdiv = env_int("PASTA_X_SUBDIV", 0);
    s->tune.graphs = env_int("PASTA_GRAPHS", 1);
  }
  if (env) {
    s->env = *env;
  } else {
    memset(&s->env, 0, sizeof(s->env));
    s->env.struct_size = (uint32_t)sizeof(pasta_env);
  }
  s->stream = (cudaStream_t)s->env.stream;
  s->N = N;
  s->Np = (int64_t)floor(Y_P * (double)N + 0.5);
  s->T = T;
  s->L = L;
  s->lin_L0 = L;
  s->lin_n = 0;
  int rc = PASTA_OK;
  do {
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev <= s->env.device) {
      set_error("no usable CUDA device %d (there is no CPU fallback): %s", s->env.device,
                cudaGetErrorString(cudaGetLastError()));
      rc = PASTA_ECUDA;
      break;
    }
    if ((rc = use_device(s)) != PASTA_OK) break;
    const size_t n = (size_t)N;
    if ((rc = buffer_reserve(s, &s->x, 24 * n)) || (rc = buffer_reserve(s, &s->v, 24 * n)) ||
        (rc = buffer_reserve(s, &s->F, 32 * n)) ||  // [F | e]: one allocation, see below
        (rc = buffer_reserve(s, &s->is_p, n)) || (rc = buffer_reserve(s, &s->cell_id, 4 * n)) ||
        (rc = buffer_reserve(s, &s->perm, 4 * n)) || (rc = buffer_reserve(s, &s->pos4, 16 * n + 4096)) ||
        (rc = buffer_reserve(s, &s->cxyz, 4 * n)) || (rc = buffer_reserve(s, &s->partials, 8 * 8192)) ||
        (rc = buffer_reserve(s, &s->scalars, 8 * 16)) || (rc = buffer_reserve(s, &s->counters, 8 * 32)))
      break;
    // e sits right behind F (N is fixed for the life of the simulation), so that a sharded evaluation zeroes and sums
    // forces and energies as ONE contiguous run of 4 N doubles: one memset, one collective (pasta_set_shard)
    s->e.ptr = s->F.as<char>() + 24 * n;
    s->e.bytes = 8 * n;
    {
      void* mb = nullptr;
      if (cudaHostAlloc(&mb, 64, cudaHostAllocMapped) != cudaSuccess ||
          cudaHostGetDevicePointer(reinterpret_cast<void**>(&s->list.mbox_dev), mb, 0) != cudaSuccess) {
        set_error("pinned mailbox allocation failed: %s", cudaGetErrorString(cudaGetLastError()));
        rc = PASTA_ECUDA;
        break;
      }
      memset(mb, 0, 64);
      s->list.mbox_host = reinterpret_cast<volatile unsigned long long*>(mb);
    }
    if (cudaMemsetAsync(s->counters.ptr, 0, 8 * 32, s->stream) != cudaSuccess ||
        cudaMemsetAsync(s->F.ptr, 0, 24 * n, s->stream) != cudaSuccess ||
        cudaMemsetAsync(s->e.ptr, 0, 8 * n, s->stream) != cudaSuccess ||
        cudaMemsetAsync(s->scalars.ptr, 0, 8 * 16, s->stream) != cudaSuccess) {
      set_error("cudaMemsetAsync failed: %s", cudaGetErrorString(cudaGetLastError()));
      rc = PASTA_ECUDA;
      break;
    }
    if ((rc = k3_init_state(s, seed)) != PASTA_OK) break;
  } while (0);
  if (rc != PASTA_OK) {
    pasta_destroy(reinterpret_cast<pasta_sim*>(s));
    return rc;
  }
  *out = reinterpret_cast<pasta_sim*>(s);
  return PASTA_OK;
}

int pasta_destroy(pasta_sim* sim) {
  Sim* s = reinterpret_cast<Sim*>(sim);
  if (!s) return PASTA_OK;
  cudaSetDevice(s->env.device);
  cudaStreamSynchronize(s->stream);
  graphs_destroy(s);
  if (s->pipe.up) {
    cudaStreamSynchronize(s->pipe.up);
    cudaStreamSynchronize(s->pipe.down);
    for (int b = 0; b < 2; ++b) {
      buffer_release(s, &s->pipe.in[b]);
      buffer_release(s, &s->pipe.out[b]);
      cudaEventDestroy(s->pipe.in_done[b]);
      cudaEventDestroy(s->pipe.in_taken[b]);
      cudaEventDestroy(s->pipe.out_ready[b]);
      cudaEventDestroy(s->pipe.out_done[b]);
    }
    cudaStreamDestroy(s->pipe.up);
    cudaStreamDestroy(s->pipe.down);
  }
  release_all(s);
  if (s->list.mbox_host) cudaFreeHost(const_cast<unsigned long long*>(s->list.mbox_host));
  for (cudaEvent_t e : s->evs)
    if (e) cudaEventDestroy(e);
  delete s;
  return PASTA_OK;
}

int pasta_forces(pasta_sim* sim, double* F_dev, double* pe_host) {
  Sim* s = reinterpret_cast<Sim*>(sim);
  PASTA_TRY(check_sim(s));
  PASTA_TRY(use_device(s));
  PASTA_TRY(evaluate_forces(s, true));
  if (F_dev)
    PASTA_CUDA_OK(cudaMemcpyAsync(F_dev, s->F.ptr, 24 * (size_t)s->N, cudaMemcpyDeviceToDevice, s->stream));
  if (pe_host) {
    PASTA_TRY(k3_sum(s, s->e.as<double>(), s->N, 1));
    PASTA_CUDA_OK(cudaMemcpyAsync(pe_host, s->scalars.as<double>() + 1, sizeof(double), cudaMemcpyDeviceToHost,
                                  s->stream));
    PASTA_CUDA_OK(cudaStreamSynchronize(s->stream));
  }
  return PASTA_OK;
}

int pasta_step(pasta_sim* sim, int64_t n, double dt) {
  Sim* s = reinterpret_cast<Sim*>(sim);
  PASTA_TRY(check_sim(s));
  if (n < 0 || !(dt > 0.0)) {
    set_error("pasta_step: need n >= 0 and dt > 0");
    return PASTA_EINVAL;
  }
  PASTA_TRY(use_device(s));
  const double sc = s->prm.scale_per_step;
  const bool energy = s->prm.energy_every_step != 0;
  if (n > 0 && !s->forces_valid) PASTA_TRY(evaluate_forces(s, energy));
  for (int64_t k = 0; k < n; ++k) {
    const double L_old = s->L;
    const bool linear = s->prm.xi_dot > 0.0;
    const double L_new = linear ? s->lin_L0 * (1.0 + s->prm.xi_dot * (dt * (double)(s->lin_n + 1))) : sc * s->L;
    if (s->prm.r_c > 0.5 * L_new) {
      set_error("pasta_step: box side %g would fall below 2 r_c", L_new);
      return PASTA_EINVAL;
    }
    PASTA_TRY(check_box_side(s->prm, L_new, "pasta_step"));
    s->L = L_new;
    const bool rescale = s->prm.thermostat_interval > 0 && ((s->step_count + 1) % s->prm.thermostat_interval) == 0;
    PASTA_TRY(step_once(s, dt, sc, linear ? L_old : L_new, energy, rescale));
  }
  return PASTA_OK;
}

int pasta_expand(pasta_sim* sim, double scale) {
  Sim* s = reinterpret_cast<Sim*>(sim);
  PASTA_TRY(check_sim(s));
  if (!(scale > 0.0) || s->prm.r_c > 0.5 * scale * s->L) {
    set_error("pasta_expand: need scale > 0 and scale*L >= 2 r_c");
    return PASTA_EINVAL;
  }
  PASTA_TRY(check_box_side(s->prm, scale * s->L, "pasta_expand"));
  PASTA_TRY(use_device(s));
  const double L_new = s->L * scale;
  PASTA_TRY(k3_wrap_scale(s, scale, L_new));
  s->list.valid = false;
  s->no_lists = false;  // another box: lists get another try
  s->L = L_new;
  s->lin_L0 = L_new;
  s->lin_n = 0;
  s->forces_valid = false;
  s->energies_valid = false;
  s->clusters_valid = false;
  return PASTA_OK;
}

int pasta_clusters(pasta_sim* sim, double r_cl, int32_t* label_dev, int64_t* n_clusters_host) {
  Sim* s = reinterpret_cast<Sim*>(sim);
  PASTA_TRY(check_sim(s));
  if (!(r_cl > 0.0) || r_cl > 0.5 * s->L) {
    set_error("pasta_clusters: need 0 < r_cl <= L/2");
    return PASTA_EINVAL;
  }
  PASTA_TRY(use_device(s));
  return k4_clusters(s, r_cl, 0.0, label_dev, n_clusters_host);
}

int pasta_clusters_mst(pasta_sim* sim, double r_pp, double r_np, int32_t* label_dev, int64_t* n_clusters_host) {
  Sim* s = reinterpret_cast<Sim*>(sim);
  PASTA_TRY(check_sim(s));
  if (!(r_np > 0.0) || !(r_pp >= r_np) || r_pp > 0.5 * s->L) {
    set_error("pasta_clusters_mst: need 0 < r_np <= r_pp <= L/2");
    return PASTA_EINVAL;
  }
  PASTA_TRY(use_device(s));
  return k4_clusters(s, r_pp, r_np, label_dev, n_clusters_host);
}

int pasta_cluster_sizes(pasta_sim* sim, int32_t* A_dev, int32_t* Z_dev) {
  Sim* s = reinterpret_cast<Sim*>(sim);
  PASTA_TRY(check_sim(s));
  if (!s->clusters_valid) {
    set_error("pasta_cluster_sizes: call pasta_clusters first (positions changed since)");
    return PASTA_ESTATE;
  }
  PASTA_TRY(use_device(s));
  if (A_dev) PASTA_CUDA_OK(cudaMemcpyAsync(A_dev, s->cl_A.ptr, 4 * (size_t)s->N, cudaMemcpyDeviceToDevice, s->stream));
  if (Z_dev) PASTA_CUDA_OK(cudaMemcpyAsync(Z_dev, s->cl_Z.ptr, 4 * (size_t)s->N, cudaMemcpyDeviceToDevice, s->stream));
  return PASTA_OK;
}

int pasta_composition(pasta_sim* sim, int32_t a_min, double* out6_host) {
  Sim* s = reinterpret_cast<Sim*>(sim);
  PASTA_TRY(check_sim(s));
  if (!out6_host) {
    set_error("out6_host is NULL");
    return PASTA_EINVAL;
  }
  if (!s->clusters_valid) {
    set_error("pasta_composition: call pasta_clusters first (positions changed since)");
    return PASTA_ESTATE;
  }
  PASTA_TRY(use_device(s));
  return k4_composition(s, a_min, out6_host);
}

int pasta_get_state(pasta_sim* sim, double* x_dev, double* v_dev, uint8_t* is_proton_dev, double* L_host,
                    int64_t* step_host) {
  Sim* s = reinterpret_cast<Sim*>(sim);
  PASTA_TRY(check_sim(s));
  PASTA_TRY(use_device(s));
  const size_t n = (size_t)s->N;
  if (x_dev) PASTA_CUDA_OK(cudaMemcpyAsync(x_dev, s->x.ptr, 24 * n, cudaMemcpyDeviceToDevice, s->stream));
  if (v_dev) PASTA_CUDA_OK(cudaMemcpyAsync(v_dev, s->v.ptr, 24 * n, cudaMemcpyDeviceToDevice, s->stream));
  if (is_proton_dev) PASTA_CUDA_OK(cudaMemcpyAsync(is_proton_dev, s->is_p.ptr, n, cudaMemcpyDeviceToDevice, s->stream));
  if (L_host) *L_host = s->L;
  if (step_host) *step_host = s->step_count;
  if (L_host || step_host) PASTA_CUDA_OK(cudaStreamSynchronize(s->stream));
  return PASTA_OK;
}

static int after_set_state(Sim* s, bool have_is_p, bool have_F, double L) {
  s->list.valid = false;
  s->no_lists = false;  // a new configuration: it may be dilute where the last one was too dense for lists
  s->L = L;
  s->lin_L0 = L;
  s->lin_n = 0;
  PASTA_TRY(k3_wrap_scale(s, 1.0, L));
  if (have_is_p) {
    PASTA_TRY(k3_count_protons(s));  // the sorted layout needs the new proton count on the host
    s->state_gen += 1;               // ... and a captured step was built for the old one
  }
  s->forces_valid = have_F;
  s->energies_valid = false;
  s->clusters_valid = false;
  return PASTA_OK;
}

int pasta_set_state(pasta_sim* sim, const double* x_dev, const double* v_dev, const uint8_t* is_proton_dev,
                    const double* F_dev, double L) {
  Sim* s = reinterpret_cast<Sim*>(sim);
  PASTA_TRY(check_sim(s));
  if (!(L > 0.0) || s->prm.r_c > 0.5 * L) {
    set_error("pasta_set_state: need L >= 2 r_c");
    return PASTA_EINVAL;
  }
  PASTA_TRY(check_box_side(s->prm, L, "pasta_set_state"));
  PASTA_TRY(use_device(s));
  const size_t n = (size_t)s->N;
  if (x_dev) PASTA_CUDA_OK(cudaMemcpyAsync(s->x.ptr, x_dev, 24 * n, cudaMemcpyDeviceToDevice, s->stream));
  if (v_dev) PASTA_CUDA_OK(cudaMemcpyAsync(s->v.ptr, v_dev, 24 * n, cudaMemcpyDeviceToDevice, s->stream));
  if (is_proton_dev) PASTA_CUDA_OK(cudaMemcpyAsync(s->is_p.ptr, is_proton_dev, n, cudaMemcpyDeviceToDevice, s->stream));
  if (F_dev) PASTA_CUDA_OK(cudaMemcpyAsync(s->F.ptr, F_dev, 24 * n, cudaMemcpyDeviceToDevice, s->stream));
  return after_set_state(s, is_proton_dev != nullptr, F_dev != nullptr, L);
}

int pasta_set_state_host(pasta_sim* sim, const double* x_host, const double* v_host, const uint8_t* is_proton_host,
                         const double* F_host, double L) {
  Sim* s = reinterpret_cast<Sim*>(sim);
  PASTA_TRY(check_sim(s));
  if (!(L > 0.0) || s->prm.r_c > 0.5 * L) {
    set_error("pasta_set_state_host: need L >= 2 r_c");
    return PASTA_EINVAL;
  }
  PASTA_TRY(check_box_side(s->prm, L, "pasta_set_state_host"));
  PASTA_TRY(use_device(s));
  const size_t n = (size_t)s->N;
  if (x_host) PASTA_CUDA_OK(cudaMemcpyAsync(s->x.ptr, x_host, 24 * n, cudaMemcpyHostToDevice, s->stream));
  if (v_host) PASTA_CUDA_OK(cudaMemcpyAsync(s->v.ptr, v_host, 24 * n, cudaMemcpyHostToDevice, s->stream));
  if (is_proton_host) PASTA_CUDA_OK(cudaMemcpyAsync(s->is_p.ptr, is_proton_host, n, cudaMemcpyHostToDevice, s->stream));
  if (F_host) PASTA_CUDA_OK(cudaMemcpyAsync(s->F.ptr, F_host, 24 * n, cudaMemcpyHostToDevice, s->stream));
  return after_set_state(s, is_proton_host != nullptr, F_host != nullptr, L);
}

int pasta_get_state_host(pasta_sim* sim, double* x_host, double* v_host, double* F_host, double* L_host,
                         int64_t* step_host) {
  Sim* s = reinterpret_cast<Sim*>(sim);
  PASTA_TRY(check_sim(s));
  PASTA_TRY(use_device(s));
  const size_t n = (size_t)s->N;
  if (F_host && !s->forces_valid) PASTA_TRY(evaluate_forces(s, s->prm.energy_every_step != 0));
  if (x_host) PASTA_CUDA_OK(cudaMemcpyAsync(x_host, s->x.ptr, 24 * n, cudaMemcpyDeviceToHost, s->stream));
  if (v_host) PASTA_CUDA_OK(cudaMemcpyAsync(v_host, s->v.ptr, 24 * n, cudaMemcpyDeviceToHost, s->stream));
  if (F_host) PASTA_CUDA_OK(cudaMemcpyAsync(F_host, s->F.ptr, 24 * n, cudaMemcpyDeviceToHost, s->stream));
  if (L_host) *L_host = s->L;
  if (step_host) *step_host = s->step_count;
  PASTA_CUDA_OK(cudaStreamSynchronize(s->stream));
  return PASTA_OK;
}

static int pipe_setup(Sim* s) {
  Sim::HostPipe& p = s->pipe;
  if (p.up) return PASTA_OK;
  PASTA_CUDA_OK(cudaStreamCreateWithFlags(&p.up, cudaStreamNonBlocking));
  PASTA_CUDA_OK(cudaStreamCreateWithFlags(&p.down, cudaStreamNonBlocking));
  for (int b = 0; b < 2; ++b) {
    PASTA_TRY(buffer_reserve(s, &p.in[b], 72 * (size_t)s->N));
    PASTA_TRY(buffer_reserve(s, &p.out[b], 72 * (size_t)s->N));
    PASTA_CUDA_OK(cudaEventCreateWithFlags(&p.in_done[b], cudaEventDisableTiming));
    PASTA_CUDA_OK(cudaEventCreateWithFlags(&p.in_taken[b], cudaEventDisableTiming));
    PASTA_CUDA_OK(cudaEventCreateWithFlags(&p.out_ready[b], cudaEventDisableTiming));
    PASTA_CUDA_OK(cudaEventCreateWithFlags(&p.out_done[b], cudaEventDisableTiming));
  }
  return PASTA_OK;
}

int pasta_set_state_host_async(pasta_sim* sim, const double* x_host, const double* v_host, const double* F_host, double L) {
  Sim* s = reinterpret_cast<Sim*>(sim);
  PASTA_TRY(check_sim(s));
  if (!x_host || !v_host || !(L > 0.0) || s->prm.r_c > 0.5 * L) {
    set_error("pasta_set_state_host_async: need x, v and L >= 2 r_c");
    return PASTA_EINVAL;
  }
  PASTA_TRY(check_box_side(s->prm, L, "pasta_set_state_host_async"));
  PASTA_TRY(use_device(s));
  PASTA_TRY(pipe_setup(s));
  Sim::HostPipe& p = s->pipe;
  const int b = (int)(p.n_in & 1);
  const size_t n = 24 * (size_t)s->N;
  char* st = p.in[b].as<char>();
  // The host buffers of the set before last may be refilled as soon as this call returns (pasta.h).  Its copies sit on
  // the upload stream behind a wait for the simulation's stream, so they may not even have started: wait for them
  // here, on the host.  (That set used this same slot b, and the pipeline stays two uploads deep.)
  if (p.n_in >= 2) PASTA_CUDA_OK(cudaEventSynchronize(p.in_done[b]));
  // upload stream: the staging buffer is free once the simulation's stream has taken the upload before last
  if (p.n_in >= 2) PASTA_CUDA_OK(cudaStreamWaitEvent(p.up, p.in_taken[b], 0));
  PASTA_CUDA_OK(cudaMemcpyAsync(st, x_host, n, cudaMemcpyHostToDevice, p.up));
  PASTA_CUDA_OK(cudaMemcpyAsync(st + n, v_host, n, cudaMemcpyHostToDevice, p.up));
  if (F_host) PASTA_CUDA_OK(cudaMemcpyAsync(st + 2 * n, F_host, n, cudaMemcpyHostToDevice, p.up));
  PASTA_CUDA_OK(cudaEventRecord(p.in_done[b], p.up));
  // simulation's stream: take the state over
  PASTA_CUDA_OK(cudaStreamWaitEvent(s->stream, p.in_done[b], 0));
  PASTA_CUDA_OK(cudaMemcpyAsync(s->x.ptr, st, n, cudaMemcpyDeviceToDevice, s->stream));
  PASTA_CUDA_OK(cudaMemcpyAsync(s->v.ptr, st + n, n, cudaMemcpyDeviceToDevice, s->stream));
  if (F_host) PASTA_CUDA_OK(cudaMemcpyAsync(s->F.ptr, st + 2 * n, n, cudaMemcpyDeviceToDevice, s->stream));
  PASTA_CUDA_OK(cudaEventRecord(p.in_taken[b], s->stream));
  p.n_in += 1;
  return after_set_state(s, false, F_host != nullptr, L);
}

int pasta_get_state_host_async(pasta_sim* sim, double* x_host, double* v_host, double* F_host, double* L_host,
                               int64_t* step_host) {
  Sim* s = reinterpret_cast<Sim*>(sim);
  PASTA_TRY(check_sim(s));
  PASTA_TRY(use_device(s));
  PASTA_TRY(pipe_setup(s));
  Sim::HostPipe& p = s->pipe;
  const int b = (int)(p.n_out & 1);
  const size_t n = 24 * (size_t)s->N;
  char* st = p.out[b].as<char>();
  if (F_host && !s->forces_valid) PASTA_TRY(evaluate_forces(s, s->prm.energy_every_step != 0));
  // simulation's stream: snapshot (the staging buffer is free once the download before last has left it)
  if (p.n_out >= 2) PASTA_CUDA_OK(cudaStreamWaitEvent(s->stream, p.out_done[b], 0));
  if (x_host) PASTA_CUDA_OK(cudaMemcpyAsync(st, s->x.ptr, n, cudaMemcpyDeviceToDevice, s->stream));
  if (v_host) PASTA_CUDA_OK(cudaMemcpyAsync(st + n, s->v.ptr, n, cudaMemcpyDeviceToDevice, s->stream));
  if (F_host) PASTA_CUDA_OK(cudaMemcpyAsync(st + 2 * n, s->F.ptr, n, cudaMemcpyDeviceToDevice, s->stream));
  PASTA_CUDA_OK(cudaEventRecord(p.out_ready[b], s->stream));
  // download stream
  PASTA_CUDA_OK(cudaStreamWaitEvent(p.down, p.out_ready[b], 0));
  if (x_host) PASTA_CUDA_OK(cudaMemcpyAsync(x_host, st, n, cudaMemcpyDeviceToHost, p.down));
  if (v_host) PASTA_CUDA_OK(cudaMemcpyAsync(v_host, st + n, n, cudaMemcpyDeviceToHost, p.down));
  if (F_host) PASTA_CUDA_OK(cudaMemcpyAsync(F_host, st + 2 * n, n, cudaMemcpyDeviceToHost, p.down));
  PASTA_CUDA_OK(cudaEventRecord(p.out_done[b], p.down));
  p.n_out += 1;
  if (L_host) *L_host = s->L;
  if (step_host) *step_host = s->step_count;
  return PASTA_OK;
}

int pasta_host_sync(pasta_sim* sim) {
  Sim* s = reinterpret_cast<Sim*>(sim);
  PASTA_TRY(check_sim(s));
  PASTA_TRY(use_device(s));
  PASTA_CUDA_OK(cudaStreamSynchronize(s->stream));
  if (s->pipe.up) PASTA_CUDA_OK(cudaStreamSynchronize(s->pipe.up));
  if (s->pipe.down) PASTA_CUDA_OK(cudaStreamSynchronize(s->pipe.down));
  return PASTA_OK;
}

int pasta_ncell(pasta_sim* sim, int32_t* ncell_side_host) {
  Sim* s = reinterpret_cast<Sim*>(sim);
  PASTA_TRY(check_sim(s));
  if (!ncell_side_host) {
    set_error("ncell_side_host is NULL");
    return PASTA_EINVAL;
  }
  *ncell_side_host = make_grid(s->L, s->prm.r_c, s->prm.cell_subdiv).ncell;
  return PASTA_OK;
}

int pasta_cells(pasta_sim* sim, int32_t* cell_id_dev, int32_t* cell_start_dev, int32_t* ncell_side_host) {
  Sim* s = reinterpret_cast<Sim*>(sim);
  PASTA_TRY(check_sim(s));
  PASTA_TRY(use_device(s));
  PASTA_TRY(k1_export_cells(s, cell_id_dev, cell_start_dev));
  if (ncell_side_host) *ncell_side_host = make_grid(s->L, s->prm.r_c, s->prm.cell_subdiv).ncell;
  return PASTA_OK;
}

int pasta_force_grid(pasta_sim* sim, int32_t* out4_host) {
  Sim* s = reinterpret_cast<Sim*>(sim);
  PASTA_TRY(check_sim(s));
  if (!out4_host) {
    set_error("out4_host is NULL");
    return PASTA_EINVAL;
  }
  GridPair g;
  Grid gr[2];
  k1_grids(s, false, gr, &g);
  for (int sp = 0; sp < 2; ++sp) {
    out4_host[2 * sp + 0] = g.ncell[sp];
    out4_host[2 * sp + 1] = g.ncx[sp];
  }
  return PASTA_OK;
}

int pasta_force_cells(pasta_sim* sim, int32_t* bin_dev, int32_t* bin_start_dev, int32_t* perm_dev) {
  Sim* s = reinterpret_cast<Sim*>(sim);
  PASTA_TRY(check_sim(s));
  PASTA_TRY(use_device(s));
  if (s->tune.force_variant == 1) {
    set_error("pasta_force_cells: PASTA_FORCE_VARIANT=1 runs on the one isotropic grid that pasta_cells reports");
    return PASTA_EINVAL;
  }
  // the list of the CURRENT positions, built by exactly the kernels a force evaluation runs
  PASTA_TRY(k1_build(s));
  const size_t n = (size_t)s->N;
  const size_t nbins = (size_t)(s->grid_sp[0].nc3 + s->grid_sp[1].nc3);
  if (bin_dev) PASTA_CUDA_OK(cudaMemcpyAsync(bin_dev, s->cell_id.ptr, 4 * n, cudaMemcpyDeviceToDevice, s->stream));
  if (bin_start_dev)
    PASTA_CUDA_OK(cudaMemcpyAsync(bin_start_dev, s->bin_start.ptr, 4 * (nbins + 1), cudaMemcpyDeviceToDevice, s->stream));
  if (perm_dev) PASTA_CUDA_OK(cudaMemcpyAsync(perm_dev, s->perm.ptr, 4 * n, cudaMemcpyDeviceToDevice, s->stream));
  return PASTA_OK;
}

int pasta_list_stats(pasta_sim* sim, int64_t* out2_host) {
  Sim* s = reinterpret_cast<Sim*>(sim);
  PASTA_TRY(check_sim(s));
  if (!out2_host) {
    set_error("out2_host is NULL");
    return PASTA_EINVAL;
  }
  out2_host[0] = s->n_force_evals;
  out2_host[1] = s->n_list_builds;
  return PASTA_OK;
}

int pasta_energy(pasta_sim* sim, double* ke_host, double* pe_host) {
  Sim* s = reinterpret_cast<Sim*>(sim);
  PASTA_TRY(check_sim(s));
  PASTA_TRY(use_device(s));
  if (pe_host) {
    if (!s->forces_valid || !s->energies_valid) PASTA_TRY(evaluate_forces(s, true));
    PASTA_TRY(k3_sum(s, s->e.as<double>(), s->N, 1));
    PASTA_CUDA_OK(cudaMemcpyAsync(pe_host, s->scalars.as<double>() + 1, sizeof(double), cudaMemcpyDeviceToHost,
                                  s->stream));
  }
  if (ke_host) PASTA_TRY(k3_kinetic(s, ke_host));
  PASTA_CUDA_OK(cudaStreamSynchronize(s->stream));
  return PASTA_OK;
}

int pasta_particle_energies(pasta_sim* sim, double* e_dev) {
  Sim* s = reinterpret_cast<Sim*>(sim);
  PASTA_TRY(check_sim(s));
  if (!e_dev) {
    set_error("e_dev is NULL");
    return PASTA_EINVAL;
  }
  PASTA_TRY(use_device(s));
  if (!s->forces_valid || !s->energies_valid) PASTA_TRY(evaluate_forces(s, true));
  PASTA_CUDA_OK(cudaMemcpyAsync(e_dev, s->e.ptr, 8 * (size_t)s->N, cudaMemcpyDeviceToDevice, s->stream));
  return PASTA_OK;
}

int pasta_pair_count(pasta_sim* sim, int64_t* ordered_pairs_host) {
  Sim* s = reinterpret_cast<Sim*>(sim);
  PASTA_TRY(check_sim(s));
  if (!ordered_pairs_host) {
    set_error("ordered_pairs_host is NULL");
    return PASTA_EINVAL;
  }
  PASTA_TRY(use_device(s));
  PASTA_TRY(k1_build(s, true));  // the counting kernel walks one common grid
  return k2_pair_count(s, ordered_pairs_host, nullptr);
}

int pasta_pair_counts(pasta_sim* sim, int64_t* out2_host) {
  Sim* s = reinterpret_cast<Sim*>(sim);
  PASTA_TRY(check_sim(s));
  if (!out2_host) {
    set_error("out2_host is NULL");
    return PASTA_EINVAL;
  }
  PASTA_TRY(use_device(s));
  PASTA_TRY(k1_build(s, true));
  return k2_pair_count(s, out2_host, out2_host + 1);
}

int pasta_force_stats(pasta_sim* sim, int64_t* out3_host) {
  Sim* s = reinterpret_cast<Sim*>(sim);
  PASTA_TRY(check_sim(s));
  if (!out3_host) {
    set_error("out3_host is NULL");
    return PASTA_EINVAL;
  }
  if (s->tune.force_variant == 1) {
    set_error("pasta_force_stats: only the chunk pair kernel keeps these statistics (PASTA_FORCE_VARIANT=1 is set)");
    return PASTA_EINVAL;
  }
  PASTA_TRY(use_device(s));
  const bool no_lists = s->no_lists;
  s->no_lists = true;  // the statistics are the chunk kernel's: sort on its own grids even where lists would be used
  int rc = k1_build(s);
  s->no_lists = no_lists;
  PASTA_TRY(rc);
  // The statistics are those of ONE complete evaluation by the chunk kernel: every target, whatever window
  // pasta_set_shard last left behind (a sharded evaluation recomputes its window each time).
  s->shard.slot_lo = 0;
  s->shard.slot_hi = 0x7fffffff;
  PASTA_TRY(k2_chunk_forces(s, true, true));
  // F and e now hold every term the chunk kernel computes, for every particle, and on every rank alike: they ARE the
  // forces of this configuration -- unless the Coulomb term comes from a kernel of its own (coulomb_all_pairs), which
  // did not run: then they are a by-product that nobody may use, and the next consumer re-evaluates.
  s->forces_valid = s->energies_valid = !s->prm.coulomb_all_pairs;
  unsigned long long h[3];
  PASTA_CUDA_OK(cudaMemcpyAsync(h, s->counters.as<unsigned long long>() + 10, sizeof(h), cudaMemcpyDeviceToHost,
                                s->stream));
  PASTA_CUDA_OK(cudaStreamSynchronize(s->stream));
  for (int k = 0; k < 3; ++k) out3_host[k] = (int64_t)h[k];
  return PASTA_OK;
}

int pasta_set_timing(pasta_sim* sim, int32_t enable) {
  Sim* s = reinterpret_cast<Sim*>(sim);
  PASTA_TRY(check_sim(s));
  timing_collect(s);
  s->timing = enable != 0;
  s->ms_acc[0] = s->ms_acc[1] = s->ms_acc[2] = 0.0;
  s->n_timed = 0;
  return PASTA_OK;
}

int pasta_get_timing(pasta_sim* sim, double* ms3_host, int64_t* n_force_evals_host) {
  Sim* s = reinterpret_cast<Sim*>(sim);
  PASTA_TRY(check_sim(s));
  PASTA_TRY(use_device(s));
  timing_collect(s);
  if (ms3_host)
    for (int k = 0; k < 3; ++k) ms3_host[k] = s->ms_acc[k];
  if (n_force_evals_host) *n_force_evals_host = s->n_timed;
  s->ms_acc[0] = s->ms_acc[1] = s->ms_acc[2] = 0.0;
  s->n_timed = 0;
  return PASTA_OK;
}

int64_t pasta_launch_count(const pasta_sim* sim) {
  const Sim* s = reinterpret_cast<const Sim*>(sim);
  return s ? s->launches : 0;
}

int pasta_set_shard(pasta_sim* sim, int32_t rank, int32_t world, pasta_allreduce_fn allreduce, void* user) {
  Sim* s = reinterpret_cast<Sim*>(sim);
  PASTA_TRY(check_sim(s));
  if (world < 1 || rank < 0 || rank >= world || (world > 1 && !allreduce)) {
    set_error("pasta_set_shard: need world >= 1, 0 <= rank < world and an allreduce callback when world > 1");
    return PASTA_EINVAL;
  }
  s->shard.rank = rank;
  s->shard.world = world;
  s->shard.allreduce = allreduce;
  s->shard.user = user;
  s->forces_valid = false;  // whatever F holds was computed under the old partition
  s->energies_valid = false;
  return PASTA_OK;
}

int pasta_shard_bounds(int64_t N, int64_t Np, double cost_p, double cost_n, int32_t world, int64_t* bounds_host) {
  if (N <= 0 || Np < 0 || Np > N || world < 1 || !(cost_p > 0.0) || !(cost_n > 0.0) || !bounds_host) {
    set_error("pasta_shard_bounds: need N > 0, 0 <= Np <= N, world >= 1, positive costs and a bounds array");
    return PASTA_EINVAL;
  }
  // cumulative cost of the sorted slots [0, t): protons first, then neutrons; rank r starts at the first slot whose
  // cumulative cost reaches r / world of the total
  const double total = cost_p * (double)Np + cost_n * (double)(N - Np);
  bounds_host[0] = 0;
  for (int32_t r = 1; r < world; ++r) {
    const double want = total * (double)r / (double)world;
    const double in_p = cost_p * (double)Np;
    double t = want <= in_p ? want / cost_p : (double)Np + (want - in_p) / cost_n;
    int64_t b = (int64_t)floor(t + 0.5);
    b = b < bounds_host[r - 1] ? bounds_host[r - 1] : (b > N ? N : b);
    bounds_host[r] = b;
  }
  bounds_host[world] = N;
  return PASTA_OK;
}

int pasta_shard_costs(const pasta_sim* sim, double* out2_host) {
  const Sim* s = reinterpret_cast<const Sim*>(sim);
  PASTA_TRY(check_sim(s));
  if (!out2_host) {
    set_error("out2_host is NULL");
    return PASTA_EINVAL;
  }
  // candidates within the reach of a pass (a sphere's worth at uniform density) times the cost of evaluating one:
  // a proton-proton candidate (screened Coulomb: 21 packed FP32 + 6 MUFU) costs about 1.64 np/nn candidates (13 + 2)
  const double sigma = sqrt(1.4426950408889634074 / (2.0 * s->prm.Lambda));
  double r_n = s->prm.r_nuc > 0.0 ? s->prm.r_nuc : s->prm.r_c;
  if (s->prm.skip_exact_zeros && sigma * r_n > 11.2472) r_n = 11.2472 / sigma;
  const double vp = s->prm.r_c * s->prm.r_c * s->prm.r_c, vn = r_n * r_n * r_n;
  const double np = (double)s->Np, nn = (double)(s->N - s->Np);
  out2_host[0] = 1.64 * np * vp + nn * vn + 1.0;
  out2_host[1] = (np + nn) * vn + 1.0;
  return PASTA_OK;
}

int64_t pasta_graph_replays(const pasta_sim* sim) {
  const Sim* s = reinterpret_cast<const Sim*>(sim);
  return s ? s->graph.replays : 0;
}

}  // extern "C"
