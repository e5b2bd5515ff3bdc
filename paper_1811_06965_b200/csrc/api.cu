// api.cu - the C ABI of include/gpipe.h: argument validation, handle life cycle, parameter
// access, tracker and trace read-out.  Never throws, never aborts across the boundary.
#include <stdio.h>
#include <string.h>

#include <new>
#include <string>
#include <vector>

#include "engine.h"

using namespace gp;

static thread_local std::string g_err;

struct gpipe {
  Engine e;
};

void gpipe_set_error_(const std::string &s) { g_err = s; }

static int fail(int code, const std::string &msg) {
  g_err = msg;
  return code;
}
static int cuda_fail(cudaError_t e, const char *where) {
  g_err = std::string(where) + ": " + cudaGetErrorName(e) + " (" + cudaGetErrorString(e) + ")" + watchdog_describe();
  return GPIPE_ECUDA;
}
#define API_CUDA(x, where)                            \
  do {                                                \
    cudaError_t e__ = (x);                            \
    if (e__ != cudaSuccess) return cuda_fail(e__, where); \
  } while (0)

#if GP_PROBES
static int env_int(const char *name, int dflt) {
  const char *v = getenv(name);
  return v && *v ? atoi(v) : dflt;
}
#endif

// fills the shape fields of an Engine from the spec; no CUDA calls
static int configure(Engine &e, const gpipe_layer_spec *spec, int K, int M, int remat, int64_t n_seqs,
                     const int32_t *cell_lo = nullptr, int n_dec = 0, float logit_clip = 0.f) {
  if (!spec) return fail(GPIPE_EINVAL, "spec is NULL");
  e.spec = *spec;
  e.n_dec = n_dec;
  e.n_enc = spec->n_layers - n_dec;
  e.logit_clip = logit_clip;
  e.dt = spec->dtype;
  if (e.dt != GPIPE_DTYPE_FP32 && e.dt != GPIPE_DTYPE_BF16) return fail(GPIPE_EINVAL, "dtype must be 0 (fp32) or 1 (bf16)");
  e.d = spec->d_model; e.H = spec->d_ffn; e.A = spec->n_heads; e.V = spec->vocab; e.S = spec->seq_len;
  if (spec->n_layers < 0 || e.d <= 0 || e.H <= 0 || e.A <= 0 || e.V <= 0 || e.S <= 0)
    return fail(GPIPE_EINVAL, "n_layers >= 0 and d_model, d_ffn, n_heads, vocab, seq_len > 0 required");
  e.dh = spec->d_head ? spec->d_head : e.d / e.A;
  if (e.dh != 16 && e.dh != 32 && e.dh != 64 && e.dh != 128) return fail(GPIPE_EINVAL, "d_head must be 16, 32, 64 or 128");
  e.da = e.A * e.dh;
  if (e.d % 4 || e.H % 4 || e.V % 4 || e.d > 2048) return fail(GPIPE_EINVAL, "d_model, d_ffn, vocab must be multiples of 4 and d_model <= 2048");
  if (e.dt == GPIPE_DTYPE_BF16 && (e.d % 8 || e.H % 32 || e.V % 8))
    return fail(GPIPE_EINVAL, "bf16 mode needs d_model and vocab multiples of 8 and d_ffn a multiple of 32 (TMA row pitches; bit-packed ReLU pattern)");
  e.eps = spec->ln_eps > 0.f ? spec->ln_eps : 1e-5f;
  int L = spec->n_layers;
  if (K < 1 || K > (L > 1 ? L : 1)) return fail(GPIPE_EINVAL, "need 1 <= K <= max(L, 1)");
  if (M < 1) return fail(GPIPE_EINVAL, "need M >= 1");
  if (n_seqs < 1 || n_seqs % M) return fail(GPIPE_EINVAL, "n_seqs must split into M equal micro-batches (PAPER.md:67)");
  e.K = K; e.M = M; e.remat = remat ? 1 : 0;
  e.n_seqs = n_seqs; e.nb = n_seqs / M; e.T_mb = e.nb * e.S; e.T_total = n_seqs * e.S;
  if (e.T_mb * (int64_t)(e.V > 3 * e.da ? e.V : 3 * e.da) >= ((int64_t)1 << 40)) return fail(GPIPE_EINVAL, "micro-batch too large");
  e.causal.assign(L, 1);
  if (spec->causal) for (int l = 0; l < L; ++l) e.causal[l] = spec->causal[l] ? 1 : 0;
  e.spec.causal = nullptr;                  // the caller's array is read here only
  if (e.encdec()) for (int l = 0; l < L; ++l) e.causal[l] = e.is_dec(l) ? 1 : 0;   // reading B1
  e.cell_lo.resize(K); e.cell_hi.resize(K);
  int base = L / K, extra = L % K;          // first L mod K cells get one more layer
  for (int k = 0; k < K; ++k) {
    e.cell_lo[k] = k * base + (k < extra ? k : extra);
    e.cell_hi[k] = e.cell_lo[k] + base + (k < extra ? 1 : 0);
  }
  if (cell_lo) {                            // explicit consecutive partition: lo[0] = 0 < ... < lo[K] = L
    if (cell_lo[0] != 0 || cell_lo[K] != L) return fail(GPIPE_EINVAL, "cell_lo[0] must be 0 and cell_lo[K] must be L");
    for (int k = 0; k < K; ++k) {
      if (L > 0 && cell_lo[k + 1] <= cell_lo[k]) return fail(GPIPE_EINVAL, "cell_lo must be strictly increasing (no empty cell)");
      e.cell_lo[k] = cell_lo[k];
      e.cell_hi[k] = cell_lo[k + 1];
    }
  }
#if GP_PROBES                                 // A/B switches of the debug build only
  e.gemm_backend = env_int("GPIPE_GEMM_SIMT", 0);
  e.replay_full = env_int("GPIPE_REPLAY_FULL", 0);
#endif
  std::string err;
  e.build_inventory(err);
  return GPIPE_OK;
}

// the optimizer kernels run per parameter home: one launch over the whole flat range, or one per cell (pipeline)
template <typename F>
static int for_each_home(Engine &e, const char *where, F &&fn) {
  if (!e.multi()) {
    Ctx c = e.ctx(0);
    API_CUDA(fn(c, e.master, e.grad, e.dt == GP_BF16 ? e.w_lp : nullptr, e.opt_ms, e.n_flat), where);
    API_CUDA(cudaStreamSynchronize(c.stream), where);
    return GPIPE_OK;
  }
  for (int k = 0; k < e.K; ++k) {
    API_CUDA(e.use(k), where);
    Ctx c = e.ctx(k);
    API_CUDA(fn(c, e.cmaster[k], e.cgrad[k], e.dt == GP_BF16 ? e.cwlp[k] : nullptr, e.copt.empty() ? nullptr : e.copt[k],
                e.cell_off[k + 1] - e.cell_off[k]), where);
  }
  for (int k = 0; k < e.K; ++k) {
    API_CUDA(e.use(k), where);
    API_CUDA(cudaStreamSynchronize(e.st(k)), where);
  }
  API_CUDA(e.use(0), where);
  return GPIPE_OK;
}

extern "C" {

const char *gpipe_last_error(void) { return g_err.c_str(); }
const char *gpipe_version(void) { return "gpipe-b200 0.1 (sm_100a)"; }

int gpipe_plan_bytes(const gpipe_layer_spec *spec, int K, int M, int remat, int64_t n_seqs, size_t *bytes_out) {
  if (!bytes_out) return fail(GPIPE_EINVAL, "bytes_out is NULL");
  Engine e;
  int rc = configure(e, spec, K, M, remat, n_seqs);
  if (rc) return rc;
  std::string err;
  rc = e.build_plan(true, err);
  if (rc) return fail(rc, err);
  *bytes_out = e.arena.used;
  return GPIPE_OK;
}

int gpipe_plan_bytes_pipeline(const gpipe_layer_spec *spec, int K, int M, int remat, int64_t n_seqs,
                              const int32_t *cell_lo, size_t *bytes_out) {
  if (!bytes_out) return fail(GPIPE_EINVAL, "bytes_out is NULL");
  Engine e;
  int rc = configure(e, spec, K, M, remat, n_seqs, cell_lo);
  if (rc) return rc;
  e.n_arenas = K;
  e.parena.assign(K, Arena());
  if (K > 1) e.boundary_staged = 1;
  std::string err;
  rc = e.build_plan(true, err);
  if (rc) return fail(rc, err);
  for (int k = 0; k < K; ++k) bytes_out[k] = e.parena[k].used;
  return GPIPE_OK;
}

static int create_impl(const gpipe_layer_spec *spec, int K, int M, int remat, int64_t n_seqs, const gpipe_env *env,
                       const int32_t *cell_lo, gpipe_t **out, const gpipe_cell_env *cells = nullptr, int flags = 0,
                       int n_dec = 0, float logit_clip = 0.f);
int gpipe_create_pipeline(const gpipe_layer_spec *spec, int K, int M, int remat, int64_t n_seqs,
                          const gpipe_cell_env *cells, const int32_t *cell_lo, int flags, gpipe_t **out) {
  if (!cells) return fail(GPIPE_EINVAL, "cells is NULL");
  return create_impl(spec, K, M, remat, n_seqs, nullptr, cell_lo, out, cells, flags);
}
int gpipe_create(const gpipe_layer_spec *spec, int K, int M, int remat, int64_t n_seqs, const gpipe_env *env, gpipe_t **out) {
  return create_impl(spec, K, M, remat, n_seqs, env, nullptr, out);
}
int gpipe_create_partitioned(const gpipe_layer_spec *spec, int K, int M, int remat, int64_t n_seqs, const gpipe_env *env,
                             const int32_t *cell_lo, gpipe_t **out) {
  if (!cell_lo) return fail(GPIPE_EINVAL, "cell_lo is NULL");
  return create_impl(spec, K, M, remat, n_seqs, env, cell_lo, out);
}
// ---- encoder-decoder T(L,H,A) ------------------------------------------------------------------
static int encdec_to_layer_spec(const gpipe_encdec_spec *s, gpipe_layer_spec *ls) {
  if (!s) return fail(GPIPE_EINVAL, "spec is NULL");
  if (s->n_enc < 1 || s->n_dec < 1) return fail(GPIPE_EINVAL, "an encoder-decoder model needs n_enc >= 1 and n_dec >= 1 (PAPER.md:160)");
  if (!(s->logit_clip >= 0.f)) return fail(GPIPE_EINVAL, "logit_clip must be >= 0 (0 = off)");
  memset(ls, 0, sizeof(*ls));
  ls->n_layers = s->n_enc + s->n_dec;
  ls->d_model = s->d_model; ls->d_ffn = s->d_ffn; ls->n_heads = s->n_heads; ls->d_head = s->d_head;
  ls->vocab = s->vocab; ls->seq_len = s->seq_len; ls->dtype = s->dtype; ls->causal = nullptr; ls->ln_eps = s->ln_eps;
  return GPIPE_OK;
}

// the cost model of gpipe_layer_costs with the decoder layers' cross-attention block: + 2 (4 d d_a) GEMM FLOPs and one
// unmasked attention over the S memory positions per token
int gpipe_layer_costs_encdec(const gpipe_encdec_spec *spec, int remat, double *layer_cost_out, double *embed_cost,
                             double *head_cost) {
  gpipe_layer_spec ls;
  int rc = encdec_to_layer_spec(spec, &ls);
  if (rc) return rc;
  Engine e;
  rc = configure(e, &ls, 1, 1, remat, 1, nullptr, spec->n_dec, spec->logit_clip);
  if (rc) return rc;
  const double d = e.d, da = e.da, H = e.H, S = e.S, V = e.V;
  const double Fg = 2.0 * (4.0 * d * da + 2.0 * d * H), Fx = 2.0 * (4.0 * d * da), Fv = 2.0 * d * V;
  const double passes_g = 3.0 + (remat ? 1.0 : 0.0), passes_a = 3.5 + (remat ? 1.0 : 0.0);
  for (int l = 0; l < ls.n_layers; ++l) {
    const bool dec = e.is_dec(l);
    const double Fa = 4.0 * S * da * (dec ? (S + 1.0) / (2.0 * S) : 1.0) + (dec ? 4.0 * S * da : 0.0);
    if (layer_cost_out) layer_cost_out[l] = passes_g * (Fg + (dec ? Fx : 0.0)) + passes_a * Fa;
  }
  if (embed_cost) *embed_cost = 0.0;
  if (head_cost) *head_cost = passes_g * Fv;
  return GPIPE_OK;
}

int gpipe_plan_bytes_encdec(const gpipe_encdec_spec *spec, int K, int M, int remat, int64_t n_seqs, const int32_t *cell_lo,
                            size_t *bytes_out) {
  if (!bytes_out) return fail(GPIPE_EINVAL, "bytes_out is NULL");
  gpipe_layer_spec ls;
  int rc = encdec_to_layer_spec(spec, &ls);
  if (rc) return rc;
  Engine e;
  rc = configure(e, &ls, K, M, remat, n_seqs, cell_lo, spec->n_dec, spec->logit_clip);
  if (rc) return rc;
  std::string err;
  rc = e.build_plan(true, err);
  if (rc) return fail(rc, err);
  *bytes_out = e.arena.used;
  return GPIPE_OK;
}

int gpipe_create_encdec(const gpipe_encdec_spec *spec, int K, int M, int remat, int64_t n_seqs, const gpipe_env *env,
                        const int32_t *cell_lo, gpipe_t **out) {
  gpipe_layer_spec ls;
  int rc = encdec_to_layer_spec(spec, &ls);
  if (rc) return rc;
  return create_impl(&ls, K, M, remat, n_seqs, env, cell_lo, out, nullptr, 0, spec->n_dec, spec->logit_clip);
}

int gpipe_plan_bytes_pipeline_encdec(const gpipe_encdec_spec *spec, int K, int M, int remat, int64_t n_seqs,
                                     const int32_t *cell_lo, size_t *bytes_out) {
  if (!bytes_out) return fail(GPIPE_EINVAL, "bytes_out is NULL");
  gpipe_layer_spec ls;
  int rc = encdec_to_layer_spec(spec, &ls);
  if (rc) return rc;
  Engine e;
  rc = configure(e, &ls, K, M, remat, n_seqs, cell_lo, spec->n_dec, spec->logit_clip);
  if (rc) return rc;
  e.n_arenas = K;
  e.parena.assign(K, Arena());
  if (K > 1) e.boundary_staged = 1;
  std::string err;
  rc = e.build_plan(true, err);
  if (rc) return fail(rc, err);
  for (int k = 0; k < K; ++k) bytes_out[k] = e.parena[k].used;
  return GPIPE_OK;
}

int gpipe_create_pipeline_encdec(const gpipe_encdec_spec *spec, int K, int M, int remat, int64_t n_seqs,
                                 const gpipe_cell_env *cells, const int32_t *cell_lo, int flags, gpipe_t **out) {
  if (!cells) return fail(GPIPE_EINVAL, "cells is NULL");
  gpipe_layer_spec ls;
  int rc = encdec_to_layer_spec(spec, &ls);
  if (rc) return rc;
  return create_impl(&ls, K, M, remat, n_seqs, nullptr, cell_lo, out, cells, flags, spec->n_dec, spec->logit_clip);
}

int gpipe_cell_range(const gpipe_t *g, int k, int32_t *lo, int32_t *hi) {
  if (!g || k < 0 || k >= g->e.K) return fail(GPIPE_EINVAL, "handle is NULL or cell index out of range");
  if (lo) *lo = g->e.cell_lo[k];
  if (hi) *hi = g->e.cell_hi[k];
  return GPIPE_OK;
}

// Cost model per token: F_g = 2 (4 d d_a + 2 d H), F_a = 4 S d_a (x (S+1)/2S when causal),
// F_v = 2 d V; a layer costs forward + backward (2 F_g + 2.5 F_a) + replay (forward again) when remat is on.
int gpipe_layer_costs(const gpipe_layer_spec *spec, int remat, double *layer_cost_out, double *embed_cost, double *head_cost) {
  Engine e;
  int rc = configure(e, spec, 1, 1, remat, 1);
  if (rc) return rc;
  const double d = e.d, da = e.da, H = e.H, S = e.S, V = e.V;
  const double Fg = 2.0 * (4.0 * d * da + 2.0 * d * H), Fv = 2.0 * d * V;
  const double passes_g = 3.0 + (remat ? 1.0 : 0.0), passes_a = 3.5 + (remat ? 1.0 : 0.0);
  for (int l = 0; l < spec->n_layers; ++l) {
    const double Fa = 4.0 * S * da * (e.causal[l] ? (S + 1.0) / (2.0 * S) : 1.0);
    if (layer_cost_out) layer_cost_out[l] = passes_g * Fg + passes_a * Fa;
  }
  if (embed_cost) *embed_cost = 0.0;                       // a gather: no FLOPs
  if (head_cost) *head_cost = passes_g * Fv;
  return GPIPE_OK;
}

// "the partitioning algorithm minimizes the variance in the estimated cost of all cells".
// The mean of the K cell costs is fixed by the total, so minimum variance = minimum sum of squares; consecutive
// cells make that an exact dynamic program: best[k][j] = min over i of best[k-1][i] + C(i, j)^2.  O(K L^2).
int gpipe_partition_min_variance(const double *layer_cost, int L, double first_extra, double last_extra, int K,
                                 int32_t *cell_lo_out) {
  if (!layer_cost || !cell_lo_out) return fail(GPIPE_EINVAL, "layer_cost and cell_lo_out are required");
  if (L < 1 || K < 1 || K > L) return fail(GPIPE_EINVAL, "need 1 <= K <= L");
  for (int l = 0; l < L; ++l)
    if (!(layer_cost[l] >= 0.0)) return fail(GPIPE_EINVAL, "layer costs must be >= 0");
  if (!(first_extra >= 0.0) || !(last_extra >= 0.0)) return fail(GPIPE_EINVAL, "extra costs must be >= 0");
  std::vector<double> pre(L + 1, 0.0);
  for (int l = 0; l < L; ++l) pre[l + 1] = pre[l] + layer_cost[l];
  auto cost = [&](int k, int i, int j) {                   // cell k = layers [i, j)
    double c = pre[j] - pre[i];
    if (k == 0) c += first_extra;
    if (k == K - 1) c += last_extra;
    return c * c;
  };
  const double INF = 1e300;
  std::vector<std::vector<double>> best(K, std::vector<double>(L + 1, INF));
  std::vector<std::vector<int>> arg(K, std::vector<int>(L + 1, -1));
  for (int j = 1; j <= L - (K - 1); ++j) { best[0][j] = cost(0, 0, j); arg[0][j] = 0; }
  for (int k = 1; k < K; ++k)
    for (int j = k + 1; j <= L - (K - 1 - k); ++j)
      for (int i = k; i < j; ++i) {                        // ascending i, strict <: ties keep the earliest boundary
        if (best[k - 1][i] >= INF) continue;
        double v = best[k - 1][i] + cost(k, i, j);
        if (v < best[k][j]) { best[k][j] = v; arg[k][j] = i; }
      }
  int j = L;
  cell_lo_out[K] = L;
  for (int k = K - 1; k >= 0; --k) { j = arg[k][j]; cell_lo_out[k] = j; }
  return GPIPE_OK;
}

static int create_impl(const gpipe_layer_spec *spec, int K, int M, int remat, int64_t n_seqs, const gpipe_env *env,
                       const int32_t *cell_lo, gpipe_t **out, const gpipe_cell_env *cells, int flags, int n_dec,
                       float logit_clip) {
  if (!out) return fail(GPIPE_EINVAL, "out is NULL");
  *out = nullptr;
  const bool pipe = cells != nullptr;
  if (!pipe && (!env || !env->arena || !env->streams)) return fail(GPIPE_EINVAL, "env, env->arena and env->streams are required");
  gpipe *g = new (std::nothrow) gpipe();
  if (!g) return fail(GPIPE_ENOMEM, "host allocation failed");
  Engine &e = g->e;
  int rc = configure(e, spec, K, M, remat, n_seqs, cell_lo, n_dec, logit_clip);
  if (rc) { delete g; return rc; }
  int dev = 0;
  cudaError_t ce = cudaGetDevice(&dev);
  if (ce != cudaSuccess) { delete g; return cuda_fail(ce, "gpipe_create: no usable CUDA device"); }
  const int dev_entry = dev;
  if (pipe) {
    e.n_arenas = K;
    e.parena.assign(K, Arena());
    e.cell_device.assign(K, dev);
    for (int k = 0; k < K; ++k) {
      if (!cells[k].arena || !cells[k].stream) { delete g; return fail(GPIPE_EINVAL, "cells[k].arena and cells[k].stream are required"); }
      if ((uintptr_t)cells[k].arena % 1024) { delete g; return fail(GPIPE_EINVAL, "arenas must be 1024-byte aligned"); }
      e.cell_device[k] = cells[k].device;
      if (cells[k].device != cells[0].device) e.multi_device = true;
      e.parena[k].base = (char *)cells[k].arena;
      e.parena[k].cap = cells[k].arena_bytes;
    }
    e.boundary_staged = (K > 1 && (e.multi_device || (flags & GPIPE_PIPE_STAGED))) ? 1 : 0;
    if (K > 1 && !e.multi_device && !(flags & GPIPE_PIPE_STAGED)) e.boundary_staged = 0;
    dev = e.cell_device[0];
  } else {
    if (env->n_streams < K) { delete g; return fail(GPIPE_EINVAL, "need one stream per cell (n_streams >= K)"); }
    if ((uintptr_t)env->arena % 1024) { delete g; return fail(GPIPE_EINVAL, "arena must be 1024-byte aligned"); }
    e.arena.base = (char *)env->arena;
    e.arena.cap = env->arena_bytes;
  }
  e.device = dev;
  if (ce == cudaSuccess) ce = cudaDeviceGetAttribute(&e.sm_count, cudaDevAttrMultiProcessorCount, dev);
  int cc_major = 0;
  if (ce == cudaSuccess) ce = cudaDeviceGetAttribute(&cc_major, cudaDevAttrComputeCapabilityMajor, dev);
  if (ce == cudaSuccess) ce = watchdog_init();
  if (ce != cudaSuccess) { delete g; return cuda_fail(ce, "gpipe_create: no usable CUDA device"); }
  if (cc_major != 10) { delete g; return fail(GPIPE_ECUDA, "gpipe_create: this library is built for sm_100a (B200) only"); }
  if (e.multi_device) {
    // neighbouring cells exchange the boundary tensors with peer copies; direct access makes them NVLink transfers
    for (int k = 0; k + 1 < K && ce == cudaSuccess; ++k) {
      const int a = e.cell_device[k], b = e.cell_device[k + 1];
      if (a == b) continue;
      for (int dir = 0; dir < 2 && ce == cudaSuccess; ++dir) {
        int can = 0;
        ce = cudaDeviceCanAccessPeer(&can, dir ? b : a, dir ? a : b);
        if (ce == cudaSuccess && can) {
          ce = cudaSetDevice(dir ? b : a);
          if (ce == cudaSuccess) ce = cudaDeviceEnablePeerAccess(dir ? a : b, 0);
          if (ce == cudaErrorPeerAccessAlreadyEnabled) { ce = cudaSuccess; cudaGetLastError(); }
        }
      }
    }
    if (ce != cudaSuccess) { cudaSetDevice(dev_entry); delete g; return cuda_fail(ce, "gpipe_create_pipeline: peer access"); }
  }
  std::string err;
  rc = e.build_plan(true, err);
  for (int k = 0; rc == GPIPE_OK && k < (pipe ? K : 1); ++k)
    if (e.ar(k).used > e.ar(k).cap)
      rc = fail(GPIPE_ENOMEM, "arena " + std::to_string(k) + " too small: need " + std::to_string(e.ar(k).used) +
                                  " bytes, have " + std::to_string(e.ar(k).cap));
  if (rc == GPIPE_OK) { rc = e.build_plan(false, err); if (rc) fail(rc, err); }
  if (rc) { cudaSetDevice(dev_entry); delete g; return rc; }
  e.streams.resize(K);
  for (int k = 0; k < K; ++k) e.streams[k] = (cudaStream_t)(pipe ? cells[k].stream : env->streams[k]);
  if (!pipe && env->n_streams >= 2 * K) {                      // a second stream per cell: weight gradients beside the chain
    e.side.resize(K);
    for (int k = 0; k < K; ++k) e.side[k] = (cudaStream_t)env->streams[K + k];
    e.side_tail.assign(K, nullptr);
  }
  e.ev_f.assign(K, std::vector<cudaEvent_t>(e.M, nullptr));
  e.ev_b.assign(K, std::vector<cudaEvent_t>(e.M, nullptr));
  e.ev_done.assign(K, nullptr);
  for (int k = 0; k < K && ce == cudaSuccess; ++k) {
    ce = e.use(k);                                             // an event lives on the device it is recorded on
    for (int m = 0; m < e.M && ce == cudaSuccess; ++m) {
      ce = cudaEventCreateWithFlags(&e.ev_f[k][m], cudaEventDisableTiming);
      if (ce == cudaSuccess) ce = cudaEventCreateWithFlags(&e.ev_b[k][m], cudaEventDisableTiming);
    }
    if (ce == cudaSuccess) ce = cudaEventCreateWithFlags(&e.ev_done[k], cudaEventDisableTiming);
  }
  if (ce == cudaSuccess) ce = e.use(0);
  if (ce == cudaSuccess) ce = cudaEventCreateWithFlags(&e.ev_in, cudaEventDisableTiming);
  if (ce == cudaSuccess) ce = cudaEventCreate(&e.ev_t0);
  if (ce == cudaSuccess) ce = cudaMallocHost((void **)&e.host_loss, sizeof(float) * (e.M + 1));
  if (ce == cudaSuccess) ce = cudaMallocHost((void **)&e.host_flag, sizeof(int) * 2);
  // parameters, gradients start at zero; positional table is built once
  for (int k = 0; k < K && ce == cudaSuccess; ++k) {
    ce = e.use(k);
    Ctx c = e.ctx(k);
    const size_t n = (size_t)(e.cell_off[k + 1] - e.cell_off[k]);
    if (ce == cudaSuccess) ce = cudaMemsetAsync(e.cmaster[k], 0, n * 4, c.stream);
    if (ce == cudaSuccess) ce = cudaMemsetAsync(e.cgrad[k], 0, n * 4, c.stream);
    if (ce == cudaSuccess && e.dt == GP_BF16) ce = cudaMemsetAsync(e.cwlp[k], 0, n * 2, c.stream);
    if (ce == cudaSuccess && e.bwd[k].splitk_ws)                // split-K counters start at zero and reset themselves
      ce = cudaMemsetAsync(e.bwd[k].splitk_ws, 0, e.splitk_ws_bytes, c.stream);
    if (ce == cudaSuccess && k == K - 1) ce = cudaMemsetAsync(e.flag_dev_last, 0, 4, c.stream);
    if (ce == cudaSuccess && k == 0) {
      ce = cudaMemsetAsync(e.flag_dev, 0, 4, c.stream);
      if (ce == cudaSuccess) ce = positional_table(c, e.pe, e.S, e.d);
    }
    if (ce == cudaSuccess) ce = cudaStreamSynchronize(c.stream);
  }
  if (e.multi_device) cudaSetDevice(dev_entry);
  if (ce != cudaSuccess) { gpipe_destroy(g); return cuda_fail(ce, "gpipe_create"); }
  *out = g;
  return GPIPE_OK;
}

void gpipe_destroy(gpipe_t *g) {
  if (!g) return;
  Engine &e = g->e;
  int dev_entry = 0;
  cudaGetDevice(&dev_entry);
  for (size_t k = 0; k < e.streams.size(); ++k) {
    e.use((int)k);
    cudaStreamSynchronize(e.streams[k]);
  }
  if (e.multi_device) cudaSetDevice(dev_entry);
  e.drop_graph();
  for (auto &v : e.ev_f) for (auto ev : v) if (ev) cudaEventDestroy(ev);
  for (auto &v : e.ev_b) for (auto ev : v) if (ev) cudaEventDestroy(ev);
  for (auto ev : e.ev_done) if (ev) cudaEventDestroy(ev);
  for (auto ev : e.ev_pool) cudaEventDestroy(ev);
  if (e.ev_in) cudaEventDestroy(e.ev_in);
  if (e.ev_t0) cudaEventDestroy(e.ev_t0);
  if (e.host_loss) cudaFreeHost(e.host_loss);
  if (e.host_flag) cudaFreeHost(e.host_flag);
  delete g;
}

int gpipe_init_params(gpipe_t *g, uint64_t seed, float std, int parity) {
  return gpipe_init_params_scaled(g, seed, std, parity, 1.f);
}

int gpipe_init_params_scaled(gpipe_t *g, uint64_t seed, float std, int parity, float ffn_scale) {
  if (!g) return fail(GPIPE_EINVAL, "handle is NULL");
  if (!(ffn_scale > 0.f)) return fail(GPIPE_EINVAL, "ffn_scale must be > 0");
  Engine &e = g->e;
  for (size_t i = 0; i < e.tensors.size(); ++i) {
    const TensorInfo &t = e.tensors[i];
    int64_t n = ((t.rows * t.cols + 63) / 64) * 64;
    float *m = e.P((int)i);
    void *w = e.dt == GP_BF16 ? e.Wl((int)i) : nullptr;
    API_CUDA(e.use(t.cell), "gpipe_init_params");
    Ctx c = e.ctx(t.cell);
    bool gamma = !t.matrix && t.name.size() >= 2 && t.name.compare(t.name.size() - 2, 2, "_g") == 0;
    cudaError_t ce;
    if (t.matrix || parity) {
      const bool ffn = t.matrix && t.name.size() >= 3 && (t.name.compare(t.name.size() - 3, 3, "w_1") == 0 ||
                                                          t.name.compare(t.name.size() - 3, 3, "w_2") == 0);
      ce = init_normal(c, e.dt, m, w, n, seed, (uint64_t)i, gamma ? 1.f : 0.f, ffn ? std * ffn_scale : std);
    } else {
      ce = fill_f32(c, m, n, gamma ? 1.f : 0.f);
      if (ce == cudaSuccess) ce = master_to_lp(c, e.dt, m, w, n, 0);
    }
    if (ce != cudaSuccess) return cuda_fail(ce, "gpipe_init_params");
    // padding elements beyond rows*cols stay harmless: nothing reads them
  }
  for (int k = 0; k < e.K; ++k) {
    API_CUDA(e.use(k), "gpipe_init_params");
    API_CUDA(cudaStreamSynchronize(e.st(k)), "gpipe_init_params");
  }
  API_CUDA(e.use(0), "gpipe_init_params");
  return GPIPE_OK;
}

static int step_common(Engine &e, float *loss_out) {
  if (!loss_out) return fail(GPIPE_EINVAL, "loss_out is NULL");
  cudaError_t ce = e.run_step(loss_out);
  if (ce != cudaSuccess) {
    for (auto s : e.streams) cudaStreamSynchronize(s);
    return cuda_fail(ce, "gpipe_step");
  }
  return GPIPE_OK;
}

int gpipe_step_encdec(gpipe_t *g, const int32_t *src, const int32_t *tgt, const int32_t *labels, float *loss_out) {
  if (!g || !src || !tgt || !labels) return fail(GPIPE_EINVAL, "handle, src, tgt and labels are required");
  Engine &e = g->e;
  if (!e.encdec()) return fail(GPIPE_EINVAL, "not an encoder-decoder handle: use gpipe_step");
  for (int64_t i = 0; i < e.T_total; ++i)
    if (src[i] < 0 || src[i] >= e.V || tgt[i] < 0 || tgt[i] >= e.V || labels[i] < 0 || labels[i] >= e.V)
      return fail(GPIPE_EINVAL, "source/target/label id outside [0, V) at flat index " + std::to_string(i));
  const size_t nb = (size_t)e.T_total * 4;
  // both id sequences go where the embedding is (cell 0), the labels where the loss is (cell K-1)
  const int kl = e.multi() ? e.K - 1 : 0;
  API_CUDA(e.use(0), "gpipe_step_encdec");
  API_CUDA(cudaMemcpyAsync(e.tok_dev, src, nb, cudaMemcpyHostToDevice, e.streams[0]), "gpipe_step_encdec H2D");
  API_CUDA(cudaMemcpyAsync(e.tgt_dev, tgt, nb, cudaMemcpyHostToDevice, e.streams[0]), "gpipe_step_encdec H2D");
  API_CUDA(e.use(kl), "gpipe_step_encdec");
  API_CUDA(cudaMemcpyAsync(e.lab_dev, labels, nb, cudaMemcpyHostToDevice, e.streams[kl]), "gpipe_step_encdec H2D");
  API_CUDA(e.use(0), "gpipe_step_encdec");
  return step_common(e, loss_out);
}

int gpipe_step_encdec_device(gpipe_t *g, const int32_t *src_dev, const int32_t *tgt_dev, const int32_t *labels_dev,
                             float *loss_out) {
  if (!g || !src_dev || !tgt_dev || !labels_dev) return fail(GPIPE_EINVAL, "handle, src, tgt and labels are required");
  Engine &e = g->e;
  if (!e.encdec()) return fail(GPIPE_EINVAL, "not an encoder-decoder handle: use gpipe_step_device");
  const int kl = e.multi() ? e.K - 1 : 0;
  const size_t nb = (size_t)e.T_total * 4;
  API_CUDA(e.use(0), "gpipe_step_encdec_device");
  Ctx c0 = e.ctx(0);
  API_CUDA(cudaMemsetAsync(e.flag_dev, 0, 4, c0.stream), "gpipe_step_encdec_device");
  API_CUDA(cudaMemcpyAsync(e.tok_dev, src_dev, nb, cudaMemcpyDefault, c0.stream), "gpipe_step_encdec_device");
  API_CUDA(cudaMemcpyAsync(e.tgt_dev, tgt_dev, nb, cudaMemcpyDefault, c0.stream), "gpipe_step_encdec_device");
  API_CUDA(check_ids(c0, e.tok_dev, e.T_total, e.V, e.flag_dev), "gpipe_step_encdec_device");
  API_CUDA(check_ids(c0, e.tgt_dev, e.T_total, e.V, e.flag_dev), "gpipe_step_encdec_device");
  API_CUDA(cudaMemcpyAsync(e.host_flag, e.flag_dev, 4, cudaMemcpyDeviceToHost, c0.stream), "gpipe_step_encdec_device");
  API_CUDA(e.use(kl), "gpipe_step_encdec_device");
  Ctx cl = e.ctx(kl);
  if (e.multi()) API_CUDA(cudaMemsetAsync(e.flag_dev_last, 0, 4, cl.stream), "gpipe_step_encdec_device");
  API_CUDA(cudaMemcpyAsync(e.lab_dev, labels_dev, nb, cudaMemcpyDefault, cl.stream), "gpipe_step_encdec_device");
  API_CUDA(check_ids(cl, e.lab_dev, e.T_total, e.V, e.flag_dev_last), "gpipe_step_encdec_device");
  API_CUDA(cudaMemcpyAsync(e.host_flag + 1, e.flag_dev_last, 4, cudaMemcpyDeviceToHost, cl.stream), "gpipe_step_encdec_device");
  API_CUDA(cudaStreamSynchronize(cl.stream), "gpipe_step_encdec_device");
  API_CUDA(e.use(0), "gpipe_step_encdec_device");
  API_CUDA(cudaStreamSynchronize(c0.stream), "gpipe_step_encdec_device");
  if (e.host_flag[0] || e.host_flag[1]) return fail(GPIPE_EINVAL, "source/target/label id outside [0, V)");
  return step_common(e, loss_out);
}

int gpipe_step(gpipe_t *g, const int32_t *tokens, const int32_t *labels, float *loss_out) {
  if (!g || !tokens || !labels) return fail(GPIPE_EINVAL, "handle, tokens and labels are required");
  Engine &e = g->e;
  if (e.encdec()) return fail(GPIPE_EINVAL, "encoder-decoder handle: use gpipe_step_encdec");
  for (int64_t i = 0; i < e.T_total; ++i)
    if (tokens[i] < 0 || tokens[i] >= e.V || labels[i] < 0 || labels[i] >= e.V)
      return fail(GPIPE_EINVAL, "token/label outside [0, V) at flat index " + std::to_string(i));
  // tokens go where the embedding is (cell 0), labels where the loss is (cell K-1)
  API_CUDA(e.use(0), "gpipe_step");
  API_CUDA(cudaMemcpyAsync(e.tok_dev, tokens, (size_t)e.T_total * 4, cudaMemcpyHostToDevice, e.streams[0]), "gpipe_step H2D");
  const int kl = e.multi() ? e.K - 1 : 0;
  API_CUDA(e.use(kl), "gpipe_step");
  API_CUDA(cudaMemcpyAsync(e.lab_dev, labels, (size_t)e.T_total * 4, cudaMemcpyHostToDevice, e.streams[kl]), "gpipe_step H2D");
  API_CUDA(e.use(0), "gpipe_step");
  return step_common(e, loss_out);
}

int gpipe_step_device(gpipe_t *g, const int32_t *tokens_dev, const int32_t *labels_dev, float *loss_out) {
  if (!g || !tokens_dev || !labels_dev) return fail(GPIPE_EINVAL, "handle, tokens and labels are required");
  Engine &e = g->e;
  if (e.encdec()) return fail(GPIPE_EINVAL, "encoder-decoder handle: use gpipe_step_encdec_device");
  const int kl = e.multi() ? e.K - 1 : 0;
  // ids move to the cells that use them (cell 0: embedding, cell K-1: loss), are range-checked there, then the step runs
  API_CUDA(e.use(0), "gpipe_step_device");
  Ctx c0 = e.ctx(0);
  API_CUDA(cudaMemsetAsync(e.flag_dev, 0, 4, c0.stream), "gpipe_step_device");
  API_CUDA(cudaMemcpyAsync(e.tok_dev, tokens_dev, (size_t)e.T_total * 4, cudaMemcpyDefault, c0.stream), "gpipe_step_device");
  API_CUDA(check_ids(c0, e.tok_dev, e.T_total, e.V, e.flag_dev), "gpipe_step_device");
  API_CUDA(cudaMemcpyAsync(e.host_flag, e.flag_dev, 4, cudaMemcpyDeviceToHost, c0.stream), "gpipe_step_device");
  API_CUDA(e.use(kl), "gpipe_step_device");
  Ctx cl = e.ctx(kl);
  if (e.multi()) API_CUDA(cudaMemsetAsync(e.flag_dev_last, 0, 4, cl.stream), "gpipe_step_device");
  API_CUDA(cudaMemcpyAsync(e.lab_dev, labels_dev, (size_t)e.T_total * 4, cudaMemcpyDefault, cl.stream), "gpipe_step_device");
  API_CUDA(check_ids(cl, e.lab_dev, e.T_total, e.V, e.flag_dev_last), "gpipe_step_device");
  API_CUDA(cudaMemcpyAsync(e.host_flag + 1, e.flag_dev_last, 4, cudaMemcpyDeviceToHost, cl.stream), "gpipe_step_device");
  API_CUDA(cudaStreamSynchronize(cl.stream), "gpipe_step_device");
  API_CUDA(e.use(0), "gpipe_step_device");
  API_CUDA(cudaStreamSynchronize(c0.stream), "gpipe_step_device");
  if (e.host_flag[0] || e.host_flag[1]) return fail(GPIPE_EINVAL, "token/label outside [0, V)");
  return step_common(e, loss_out);
}

int gpipe_apply_sgd(gpipe_t *g, float lr) {
  if (!g) return fail(GPIPE_EINVAL, "handle is NULL");
  Engine &e = g->e;
  return for_each_home(e, "gpipe_apply_sgd", [&](const Ctx &c, float *m, float *gr, void *w, float *, int64_t n) {
    return sgd_apply(c, e.dt, m, gr, w, n, lr);
  });
}

int gpipe_optimizer_slot_bytes(const gpipe_t *g, size_t *bytes_out) {
  if (!g || !bytes_out) return fail(GPIPE_EINVAL, "handle and bytes_out are required");
  *bytes_out = (size_t)g->e.n_flat * sizeof(float);
  return GPIPE_OK;
}

int gpipe_attach_optimizer_slots(gpipe_t *g, void *slots_dev, size_t bytes) {
  if (!g || !slots_dev) return fail(GPIPE_EINVAL, "handle and slots_dev are required");
  Engine &e = g->e;
  if (e.multi()) return fail(GPIPE_ENOTIMPL, "pipeline handles take one slot buffer per cell: gpipe_attach_optimizer_slots_cell");
  if (bytes < (size_t)e.n_flat * sizeof(float)) return fail(GPIPE_ENOMEM, "optimizer slots too small: need " + std::to_string((size_t)e.n_flat * 4) + " bytes");
  if ((uintptr_t)slots_dev % 16) return fail(GPIPE_EINVAL, "optimizer slots must be 16-byte aligned");
  API_CUDA(cudaMemsetAsync(slots_dev, 0, (size_t)e.n_flat * sizeof(float), e.streams[0]), "gpipe_attach_optimizer_slots");
  API_CUDA(cudaStreamSynchronize(e.streams[0]), "gpipe_attach_optimizer_slots");
  e.opt_ms = (float *)slots_dev;
  e.copt.assign(e.K, nullptr);
  for (int k = 0; k < e.K; ++k) e.copt[k] = e.opt_ms + e.cell_off[k];
  return GPIPE_OK;
}

int gpipe_attach_optimizer_slots_cell(gpipe_t *g, int k, void *slots_dev, size_t bytes) {
  if (!g || !slots_dev) return fail(GPIPE_EINVAL, "handle and slots_dev are required");
  Engine &e = g->e;
  if (k < 0 || k >= e.K) return fail(GPIPE_EINVAL, "cell index out of range");
  const size_t need = (size_t)(e.cell_off[k + 1] - e.cell_off[k]) * sizeof(float);
  if (bytes < need) return fail(GPIPE_ENOMEM, "optimizer slots too small: need " + std::to_string(need) + " bytes");
  if ((uintptr_t)slots_dev % 16) return fail(GPIPE_EINVAL, "optimizer slots must be 16-byte aligned");
  API_CUDA(e.use(k), "gpipe_attach_optimizer_slots_cell");
  API_CUDA(cudaMemsetAsync(slots_dev, 0, need, e.st(k)), "gpipe_attach_optimizer_slots_cell");
  API_CUDA(cudaStreamSynchronize(e.st(k)), "gpipe_attach_optimizer_slots_cell");
  API_CUDA(e.use(0), "gpipe_attach_optimizer_slots_cell");
  if (e.copt.empty()) e.copt.assign(e.K, nullptr);
  e.copt[k] = (float *)slots_dev;
  bool all = true;
  for (float *p : e.copt) all = all && p != nullptr;
  if (all && e.multi()) e.opt_ms = e.copt[0];             // "slots attached" marker
  return GPIPE_OK;
}

int gpipe_cell_param_count(const gpipe_t *g, int k, int64_t *n_out) {
  if (!g || !n_out || k < 0 || k >= g->e.K) return fail(GPIPE_EINVAL, "handle, n_out and a valid cell index are required");
  *n_out = g->e.cell_off[k + 1] - g->e.cell_off[k];
  return GPIPE_OK;
}

int gpipe_apply_rmsprop(gpipe_t *g, float lr, float rho, float eps) {
  if (!g) return fail(GPIPE_EINVAL, "handle is NULL");
  Engine &e = g->e;
  if (!e.opt_ms) return fail(GPIPE_EINVAL, "call gpipe_attach_optimizer_slots first");
  if (!(rho >= 0.f && rho < 1.f) || !(eps > 0.f)) return fail(GPIPE_EINVAL, "need 0 <= rho < 1 and eps > 0");
  return for_each_home(e, "gpipe_apply_rmsprop", [&](const Ctx &c, float *m, float *gr, void *w, float *ms, int64_t n) {
    return rmsprop_apply(c, e.dt, m, gr, ms, w, n, lr, rho, eps);
  });
}

// ---- data-parallel replicas -------------------------------------------------------------------
int gpipe_dp_shard(int64_t n_flat, int rank, int world, int64_t *lo, int64_t *hi) {
  if (n_flat < 0 || world < 1 || rank < 0 || rank >= world || !lo || !hi) return fail(GPIPE_EINVAL, "need n_flat >= 0, 0 <= rank < world");
  dp_shard(n_flat, rank, world, lo, hi);
  return GPIPE_OK;
}

int gpipe_dp_layout(const gpipe_t *g, int64_t *n_flat, size_t *master_off, size_t *grad_off, size_t *wlp_off) {
  if (!g) return fail(GPIPE_EINVAL, "handle is NULL");
  const Engine &e = g->e;
  if (e.multi()) return fail(GPIPE_ENOTIMPL, "data-parallel replicas of a pipeline handle are not built");
  if (n_flat) *n_flat = e.n_flat;
  if (master_off) *master_off = (size_t)((const char *)e.master - e.arena.base);
  if (grad_off) *grad_off = (size_t)((const char *)e.grad - e.arena.base);
  if (wlp_off) *wlp_off = e.dt == GP_BF16 ? (size_t)((const char *)e.w_lp - e.arena.base) : (size_t)0;
  return GPIPE_OK;
}

static int dp_apply_impl(gpipe_t *g, int rank, int world, void *const *peer_arenas, float lr, float grad_scale, int rms,
                         float rho, float eps, const char *where) {
  if (!g || !peer_arenas) return fail(GPIPE_EINVAL, "handle and peer_arenas are required");
  Engine &e = g->e;
  if (e.multi()) return fail(GPIPE_ENOTIMPL, "data-parallel replicas of a pipeline handle are not built");
  if (world < 1 || world > DpPeers::kMax || rank < 0 || rank >= world)
    return fail(GPIPE_EINVAL, "need 1 <= world <= " + std::to_string(DpPeers::kMax) + " and 0 <= rank < world");
  if (peer_arenas[rank] != (void *)e.arena.base) return fail(GPIPE_EINVAL, "peer_arenas[rank] must be this handle's own arena");
  if (rms && !e.opt_ms) return fail(GPIPE_EINVAL, "call gpipe_attach_optimizer_slots first");
  if (rms && (!(rho >= 0.f && rho < 1.f) || !(eps > 0.f))) return fail(GPIPE_EINVAL, "need 0 <= rho < 1 and eps > 0");
  DpPeers P{};
  const size_t mo = (size_t)((char *)e.master - e.arena.base), go = (size_t)((char *)e.grad - e.arena.base);
  const size_t wo = e.dt == GP_BF16 ? (size_t)((char *)e.w_lp - e.arena.base) : 0;
  for (int p = 0; p < world; ++p) {
    if (!peer_arenas[p]) return fail(GPIPE_EINVAL, "peer_arenas[" + std::to_string(p) + "] is NULL");
    char *b = (char *)peer_arenas[p];                       // same spec, K, M, n_seqs -> same plan -> same offsets
    P.master[p] = (float *)(b + mo);
    P.grad[p] = (float *)(b + go);
    P.wlp[p] = e.dt == GP_BF16 ? (void *)(b + wo) : nullptr;
  }
  P.slot = rms ? e.opt_ms : nullptr;
  Ctx c = e.ctx(0);
  API_CUDA(dp_apply(c, e.dt, P, world, rank, e.n_flat, lr, grad_scale, rms, rho, eps), where);
  API_CUDA(cudaStreamSynchronize(c.stream), where);
  return GPIPE_OK;
}

int gpipe_dp_apply_sgd(gpipe_t *g, int rank, int world, void *const *peer_arenas, float lr, float grad_scale) {
  return dp_apply_impl(g, rank, world, peer_arenas, lr, grad_scale, 0, 0.f, 1.f, "gpipe_dp_apply_sgd");
}

int gpipe_dp_apply_rmsprop(gpipe_t *g, int rank, int world, void *const *peer_arenas, float lr, float rho, float eps,
                           float grad_scale) {
  return dp_apply_impl(g, rank, world, peer_arenas, lr, grad_scale, 1, rho, eps, "gpipe_dp_apply_rmsprop");
}

// CUDA IPC plumbing for the peer arenas (one process per GPU): the handle of the ALLOCATION that contains dev_ptr and
// the offset of dev_ptr inside it; the peer opens the allocation and adds the offset.
int gpipe_ipc_export(const void *dev_ptr, unsigned char *handle_out, size_t *offset_out) {
  if (!dev_ptr || !handle_out || !offset_out) return fail(GPIPE_EINVAL, "arguments are required");
  typedef int (*GetRangeFn)(unsigned long long *, size_t *, unsigned long long);
  void *fp = nullptr;
  cudaDriverEntryPointQueryResult q;
  API_CUDA(cudaGetDriverEntryPoint("cuMemGetAddressRange", &fp, cudaEnableDefault, &q), "gpipe_ipc_export");
  if (!fp || q != cudaDriverEntryPointSuccess) return fail(GPIPE_ECUDA, "gpipe_ipc_export: cuMemGetAddressRange unavailable");
  unsigned long long base = 0;
  size_t size = 0;
  if (((GetRangeFn)fp)(&base, &size, (unsigned long long)(uintptr_t)dev_ptr) != 0)
    return fail(GPIPE_ECUDA, "gpipe_ipc_export: cuMemGetAddressRange failed (not a device allocation?)");
  cudaIpcMemHandle_t h;
  API_CUDA(cudaIpcGetMemHandle(&h, (void *)(uintptr_t)base), "gpipe_ipc_export");
  static_assert(sizeof(h) == 64, "cudaIpcMemHandle_t is 64 bytes");
  memcpy(handle_out, &h, 64);
  *offset_out = (size_t)((uintptr_t)dev_ptr - (uintptr_t)base);
  return GPIPE_OK;
}

int gpipe_ipc_open(const unsigned char *handle, void **base_out) {
  if (!handle || !base_out) return fail(GPIPE_EINVAL, "arguments are required");
  cudaIpcMemHandle_t h;
  memcpy(&h, handle, 64);
  API_CUDA(cudaIpcOpenMemHandle(base_out, h, cudaIpcMemLazyEnablePeerAccess), "gpipe_ipc_open");
  return GPIPE_OK;
}

int gpipe_ipc_close(void *base) {
  if (!base) return GPIPE_OK;
  API_CUDA(cudaIpcCloseMemHandle(base), "gpipe_ipc_close");
  return GPIPE_OK;
}

int gpipe_zero_grads(gpipe_t *g) {
  if (!g) return fail(GPIPE_EINVAL, "handle is NULL");
  Engine &e = g->e;
  return for_each_home(e, "gpipe_zero_grads", [&](const Ctx &c, float *, float *gr, void *, float *, int64_t n) {
    return cudaMemsetAsync(gr, 0, (size_t)n * 4, c.stream);
  });
}

int gpipe_num_tensors(const gpipe_t *g) { return g ? (int)g->e.tensors.size() : fail(GPIPE_EINVAL, "handle is NULL"); }

int gpipe_tensor_info(const gpipe_t *g, int i, const char **name, int64_t *rows, int64_t *cols) {
  if (!g) return fail(GPIPE_EINVAL, "handle is NULL");
  if (i < 0 || i >= (int)g->e.tensors.size()) return fail(GPIPE_EINVAL, "tensor index out of range");
  const TensorInfo &t = g->e.tensors[i];
  if (name) *name = t.name.c_str();
  if (rows) *rows = t.rows;
  if (cols) *cols = t.cols;
  return GPIPE_OK;
}

static int tensor_check(gpipe_t *g, int i, const void *p) {
  if (!g || !p) return fail(GPIPE_EINVAL, "handle and host pointer are required");
  if (i < 0 || i >= (int)g->e.tensors.size()) return fail(GPIPE_EINVAL, "tensor index out of range");
  return GPIPE_OK;
}

int gpipe_get_param(gpipe_t *g, int i, float *host_out) {
  int rc = tensor_check(g, i, host_out);
  if (rc) return rc;
  Engine &e = g->e;
  const TensorInfo &t = e.tensors[i];
  int64_t n = t.rows * t.cols;
  API_CUDA(e.use(t.cell), "gpipe_get_param");
  Ctx c = e.ctx(t.cell);
  if (e.dt == GP_BF16 && t.matrix) {
    // widen the bf16 working copy on the host
    std::string tmp((size_t)n * 2, '\0');
    API_CUDA(cudaMemcpyAsync(&tmp[0], e.Wl(i), (size_t)n * 2, cudaMemcpyDeviceToHost, c.stream), "gpipe_get_param");
    API_CUDA(cudaStreamSynchronize(c.stream), "gpipe_get_param");
    API_CUDA(e.use(0), "gpipe_get_param");
    const uint16_t *u = (const uint16_t *)tmp.data();
    for (int64_t j = 0; j < n; ++j) {
      uint32_t w = (uint32_t)u[j] << 16;
      memcpy(host_out + j, &w, 4);
    }
    return GPIPE_OK;
  }
  API_CUDA(cudaMemcpyAsync(host_out, e.P(i), (size_t)n * 4, cudaMemcpyDeviceToHost, c.stream), "gpipe_get_param");
  API_CUDA(cudaStreamSynchronize(c.stream), "gpipe_get_param");
  API_CUDA(e.use(0), "gpipe_get_param");
  return GPIPE_OK;
}

int gpipe_set_param(gpipe_t *g, int i, const float *host_in) {
  int rc = tensor_check(g, i, host_in);
  if (rc) return rc;
  Engine &e = g->e;
  const TensorInfo &t = e.tensors[i];
  int64_t n = t.rows * t.cols;
  API_CUDA(e.use(t.cell), "gpipe_set_param");
  Ctx c = e.ctx(t.cell);
  API_CUDA(cudaMemcpyAsync(e.P(i), host_in, (size_t)n * 4, cudaMemcpyHostToDevice, c.stream), "gpipe_set_param");
  if (e.dt == GP_BF16)   // RNE-round into the working copy; matrices also round the master (A12)
    API_CUDA(master_to_lp(c, e.dt, e.P(i), e.Wl(i), n, t.matrix ? 1 : 0), "gpipe_set_param");
  API_CUDA(cudaStreamSynchronize(c.stream), "gpipe_set_param");
  API_CUDA(e.use(0), "gpipe_set_param");
  return GPIPE_OK;
}

// ---- exact state access for checkpoint / resume: no rounding anywhere -------------------------------------------
int gpipe_get_master(gpipe_t *g, int i, float *host_out) {
  int rc = tensor_check(g, i, host_out);
  if (rc) return rc;
  Engine &e = g->e;
  const TensorInfo &t = e.tensors[i];
  API_CUDA(e.use(t.cell), "gpipe_get_master");
  API_CUDA(cudaMemcpyAsync(host_out, e.P(i), (size_t)(t.rows * t.cols) * 4, cudaMemcpyDeviceToHost, e.st(t.cell)), "gpipe_get_master");
  API_CUDA(cudaStreamSynchronize(e.st(t.cell)), "gpipe_get_master");
  API_CUDA(e.use(0), "gpipe_get_master");
  return GPIPE_OK;
}

int gpipe_set_master(gpipe_t *g, int i, const float *host_in) {
  int rc = tensor_check(g, i, host_in);
  if (rc) return rc;
  Engine &e = g->e;
  const TensorInfo &t = e.tensors[i];
  int64_t n = t.rows * t.cols;
  API_CUDA(e.use(t.cell), "gpipe_set_master");
  Ctx c = e.ctx(t.cell);
  API_CUDA(cudaMemcpyAsync(e.P(i), host_in, (size_t)n * 4, cudaMemcpyHostToDevice, c.stream), "gpipe_set_master");
  if (e.dt == GP_BF16)   // working copy = RNE(master); the master keeps every bit
    API_CUDA(master_to_lp(c, e.dt, e.P(i), e.Wl(i), n, 0), "gpipe_set_master");
  API_CUDA(cudaStreamSynchronize(c.stream), "gpipe_set_master");
  API_CUDA(e.use(0), "gpipe_set_master");
  return GPIPE_OK;
}

int gpipe_get_optimizer_slot(gpipe_t *g, int i, float *host_out) {
  int rc = tensor_check(g, i, host_out);
  if (rc) return rc;
  Engine &e = g->e;
  if (!e.opt_ms) return fail(GPIPE_EINVAL, "no optimizer slots attached");
  const TensorInfo &t = e.tensors[i];
  API_CUDA(e.use(t.cell), "gpipe_get_optimizer_slot");
  API_CUDA(cudaMemcpyAsync(host_out, e.Opt(i), (size_t)(t.rows * t.cols) * 4, cudaMemcpyDeviceToHost, e.st(t.cell)), "gpipe_get_optimizer_slot");
  API_CUDA(cudaStreamSynchronize(e.st(t.cell)), "gpipe_get_optimizer_slot");
  API_CUDA(e.use(0), "gpipe_get_optimizer_slot");
  return GPIPE_OK;
}

int gpipe_set_optimizer_slot(gpipe_t *g, int i, const float *host_in) {
  int rc = tensor_check(g, i, host_in);
  if (rc) return rc;
  Engine &e = g->e;
  if (!e.opt_ms) return fail(GPIPE_EINVAL, "no optimizer slots attached");
  const TensorInfo &t = e.tensors[i];
  API_CUDA(e.use(t.cell), "gpipe_set_optimizer_slot");
  API_CUDA(cudaMemcpyAsync(e.Opt(i), host_in, (size_t)(t.rows * t.cols) * 4, cudaMemcpyHostToDevice, e.st(t.cell)), "gpipe_set_optimizer_slot");
  API_CUDA(cudaStreamSynchronize(e.st(t.cell)), "gpipe_set_optimizer_slot");
  API_CUDA(e.use(0), "gpipe_set_optimizer_slot");
  return GPIPE_OK;
}

int gpipe_get_grad(gpipe_t *g, int i, float *host_out) {
  int rc = tensor_check(g, i, host_out);
  if (rc) return rc;
  Engine &e = g->e;
  const TensorInfo &t = e.tensors[i];
  API_CUDA(e.use(t.cell), "gpipe_get_grad");
  API_CUDA(cudaMemcpyAsync(host_out, e.G(i), (size_t)(t.rows * t.cols) * 4, cudaMemcpyDeviceToHost, e.st(t.cell)), "gpipe_get_grad");
  API_CUDA(cudaStreamSynchronize(e.st(t.cell)), "gpipe_get_grad");
  API_CUDA(e.use(0), "gpipe_get_grad");
  return GPIPE_OK;
}

int gpipe_peak_bytes(const gpipe_t *g, size_t *total, size_t *by_category, size_t *by_cell) {
  if (!g) return fail(GPIPE_EINVAL, "handle is NULL");
  const Engine &e = g->e;
  // pipeline handle: totals over the K arenas; by_cell[k] is then everything cell k's device holds (PAPER.md:87 is
  // stated per accelerator)
  size_t tot = 0, cat[GPIPE_NUM_CATS] = {0};
  for (int k = 0; k < (e.multi() ? e.K : 1); ++k) {
    tot += e.ar(k).used;
    for (int i = 0; i < GPIPE_NUM_CATS; ++i) cat[i] += e.ar(k).by_cat[i];
  }
  if (total) *total = tot;
  if (by_category) for (int i = 0; i < GPIPE_NUM_CATS; ++i) by_category[i] = cat[i];
  if (by_cell) for (int k = 0; k < e.K; ++k) by_cell[k] = e.multi() ? e.ar(k).used : e.arena.by_cell[k];
  return GPIPE_OK;
}

int gpipe_trace(gpipe_t *g, int enable, gpipe_trace_event *events_out, int64_t *n_events) {
  if (!g) return fail(GPIPE_EINVAL, "handle is NULL");
  Engine &e = g->e;
  e.trace_on = enable ? 1 : 0;
  if (!n_events) return GPIPE_OK;
  if (!events_out) { *n_events = (int64_t)e.trace.size(); return GPIPE_OK; }
  int64_t n = *n_events < (int64_t)e.trace.size() ? *n_events : (int64_t)e.trace.size();
  for (int64_t i = 0; i < n; ++i) {
    const TraceRec &r = e.trace[i];
    gpipe_trace_event &o = events_out[i];
    o.kind = r.kind; o.k = r.k; o.m = r.m; o.enqueue_index = r.idx;
    API_CUDA(cudaEventElapsedTime(&o.start_ms, e.ev_t0, r.e0), "gpipe_trace");
    API_CUDA(cudaEventElapsedTime(&o.end_ms, e.ev_t0, r.e1), "gpipe_trace");
  }
  *n_events = n;
  return GPIPE_OK;
}

int gpipe_kernel_timing(gpipe_t *g, int enable) {
  if (!g) return fail(GPIPE_EINVAL, "handle is NULL");
  g->e.ktiming_on = (enable & 1) ? 1 : 0;
  g->e.serial = (enable & 2) ? 1 : 0;
  for (auto &st : g->e.kstats) st = KStat();
  return GPIPE_OK;
}

int gpipe_kernel_stats(const gpipe_t *g, int cls, const char **name, int64_t *count, double *ms, double *flops, double *bytes) {
  static const char *names[KC_NUM] = {"gemm_fwd", "gemm_dgrad", "gemm_wgrad", "attn_fwd", "attn_bwd",
                                      "ln_fwd", "ln_bwd", "softmax_ce", "colsum", "embed"};
  if (!g) return fail(GPIPE_EINVAL, "handle is NULL");
  if (cls < 0 || cls >= KC_NUM) return fail(GPIPE_EINVAL, "kernel class out of range");
  const KStat &st = g->e.kstats[cls];
  if (name) *name = names[cls];
  if (count) *count = st.count;
  if (ms) *ms = st.ms;
  if (flops) *flops = st.flops;
  if (bytes) *bytes = st.bytes;
  return GPIPE_OK;
}

int64_t gpipe_launch_count(const gpipe_t *g) { return g ? g->e.launches : 0; }

int gpipe_cuda_graph(gpipe_t *g, int enable) {
  if (!g) return fail(GPIPE_EINVAL, "handle is NULL");
  Engine &e = g->e;
  for (auto s : e.streams) cudaStreamSynchronize(s);
  e.use_graph = enable ? 1 : 0;
  if (!enable) { e.drop_graph(); e.graph_state = 0; }
  else if (e.graph_state < 0) e.graph_state = 0;
  return GPIPE_OK;
}

int gpipe_cuda_graph_state(const gpipe_t *g) { return g ? (g->e.use_graph ? g->e.graph_state : 0) : fail(GPIPE_EINVAL, "handle is NULL"); }

int gpipe_debug_read(gpipe_t *g, const char *what, int layer, float *host_out, int64_t max_elems, int64_t *n_elems) {
  if (!g || !what || !host_out || !n_elems) return fail(GPIPE_EINVAL, "arguments are required");
  Engine &e = g->e;
  std::string w(what);
  const void *src = nullptr;
  int64_t n = 0;
  bool is_lp = true;
  int k = e.K - 1, li = 0;
  if (layer >= 0) {
    if (layer >= e.spec.n_layers) return fail(GPIPE_EINVAL, "layer out of range");
    for (k = 0; k < e.K; ++k) if (layer >= e.cell_lo[k] && layer < e.cell_hi[k]) break;
    li = layer - e.cell_lo[k];
  }
  Workspace &ws = e.wsp(k, 0);
  int64_t T = e.T_mb;
  if (layer >= 0) {
    LayerBuf &b = ws.layers[li];
    if (w == "a") { src = b.a; n = T * e.d; }
    else if (w == "qkv") { src = b.qkv; n = T * 3 * e.da; }
    else if (w == "o") { src = b.o; n = T * e.da; }
    else if (w == "c") { src = b.c; n = T * e.d; }
    else if (w == "h") { src = b.h; n = T * e.H; }
    else if (w == "x1") { src = b.x1; n = T * e.d; is_lp = false; }
    else if (w == "lse") { src = b.lse; n = T * e.A; is_lp = false; }
    // the bit-packed ReLU pattern [h > 0] FFN1's epilogue wrote: uint32 words, returned bit-exact in the fp32 slots
    else if (w == "hbits") { src = b.hbits; n = T * (int64_t)((e.H + 31) / 32); is_lp = false; }
  } else {
    if (w == "y") { src = ws.y; n = T * e.d; }
    else if (w == "dlogits") { src = ws.logits; n = T * e.V; }
    else if (w == "x_out") { src = ws.x_out; n = T * e.d; is_lp = false; }
  }
  if (!src) return fail(GPIPE_EINVAL, "unknown debug buffer '" + w + "'");
  if (n > max_elems) return fail(GPIPE_EINVAL, "host buffer too small: need " + std::to_string(n));
  Ctx c = e.ctx(0);
  if (is_lp && e.dt == GP_BF16) {
    std::string tmp((size_t)n * 2, '\0');
    API_CUDA(cudaMemcpy(&tmp[0], src, (size_t)n * 2, cudaMemcpyDeviceToHost), "gpipe_debug_read");
    const uint16_t *u = (const uint16_t *)tmp.data();
    for (int64_t j = 0; j < n; ++j) { uint32_t x = (uint32_t)u[j] << 16; memcpy(host_out + j, &x, 4); }
  } else {
    API_CUDA(cudaMemcpy(host_out, src, (size_t)n * 4, cudaMemcpyDeviceToHost), "gpipe_debug_read");
  }
  (void)c;
  *n_elems = n;
  return GPIPE_OK;
}

}  // extern "C"
