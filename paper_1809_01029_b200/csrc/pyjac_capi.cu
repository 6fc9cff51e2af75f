// C ABI of pyjac-b200 (include/pyjac.h): handle management, argument checking, table upload,
// kernel dispatch.  No torch types; plain pointers and sizes only.
#include <cuda_runtime.h>

#include <atomic>
#include <mutex>
#include <cstdio>
#include <cstring>
#include <new>
#include <string>
#include <vector>

#include "pyjac_internal.h"

using namespace pyjac;

namespace {
thread_local std::string g_err;
int fail(int code, const std::string& msg) { g_err = msg; return code; }
int cuda_fail(cudaError_t e, const char* what) {
  g_err = std::string(what) + ": " + cudaGetErrorString(e);
  return PYJAC_ECUDA;
}
#define CK(call) do { cudaError_t e_ = (call); if (e_ != cudaSuccess) return cuda_fail(e_, #call); } while (0)

// Scratch of pyjac_jacobian_sparse_static (include/pyjac.h): the tile counter and the finished-CTA counter of the persistent
// Jacobian kernels, in the library's own image instead of cudaMalloc'ed memory.  256 bytes (2 words used, the rest
// reserved), held by every GPU that loads the library until the process exits.  In HOST code the name g_static_sched is
// a host-side stand-in, not a device address: the address is taken with cudaGetSymbolAddress once per device, with that
// device current (static_sched_address), and only that pointer is ever passed to a kernel.
constexpr int STATIC_SCHED_WORDS = 32;
static __device__ __align__(256) unsigned long long g_static_sched[STATIC_SCHED_WORDS];
constexpr int MAX_DEVICES = 64;
std::mutex g_static_mu;
unsigned long long* g_static_addr[MAX_DEVICES] = {};
// device `dev` must be current
int static_sched_address(int dev, unsigned long long** out) {
  if (dev < 0 || dev >= MAX_DEVICES) return fail(PYJAC_ECUDA, "static scratch: device index beyond " + std::to_string(MAX_DEVICES - 1));
  std::lock_guard<std::mutex> lock(g_static_mu);
  if (!g_static_addr[dev]) {
    unsigned long long* p = nullptr;
    CK(cudaGetSymbolAddress((void**)&p, g_static_sched));
    CK(cudaMemset(p, 0, sizeof(unsigned long long) * STATIC_SCHED_WORDS));
    g_static_addr[dev] = p;
  }
  *out = g_static_addr[dev];
  return PYJAC_OK;
}

// ---- fraction <-> state conversions (Eq. 1; include/pyjac.h) ---------------------------------------
// One thread per state, the species loop inside: with the state index fastest in memory (tile > 1) every load and store
// of a warp is a contiguous run.  wr[k] = W_k / W_Ns: only ratios of molecular weights enter.
__device__ __forceinline__ int64_t conv_base(int64_t s, int64_t tile, int64_t n_e) {
  if (tile & (tile - 1)) return s;                       // tile == ld: one tile holds every state
  const int sh = __ffsll((long long)tile) - 1;
  return (((s >> sh) * n_e) << sh) + (s & (tile - 1));
}
__global__ void __launch_bounds__(256) state_from_fractions_kernel(int ns, int mode, int kind, int64_t n, int64_t tile,
                                                                   const double* __restrict__ wr, const double* __restrict__ T,
                                                                   const double* __restrict__ P, const double* __restrict__ V,
                                                                   const double* __restrict__ frac, double* __restrict__ phi,
                                                                   double* __restrict__ param) {
  const int64_t s = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (s >= n) return;
  const double* __restrict__ f = frac + conv_base(s, tile, ns);
  double* __restrict__ o = phi + conv_base(s, tile, ns + 1);
  double scale = P[s] * V[s] / (R_GAS * T[s]);            // n_tot = P V / (R T)
  if (kind == PYJAC_MASS_FRACTION) {                      // X_k = (Y_k / W_k) / sum_j (Y_j / W_j)
    double sum = 0.0;
    for (int k = 0; k < ns; ++k) sum += f[(int64_t)k * tile] / __ldg(wr + k);
    scale /= sum;
  }
  o[0] = T[s];
  o[tile] = mode == PYJAC_CONP ? V[s] : P[s];
  param[s] = mode == PYJAC_CONP ? P[s] : V[s];
  for (int k = 0; k < ns - 1; ++k) {
    const double x = kind == PYJAC_MASS_FRACTION ? f[(int64_t)k * tile] / __ldg(wr + k) : f[(int64_t)k * tile];
    o[(int64_t)(2 + k) * tile] = x * scale;
  }
}
__global__ void __launch_bounds__(256) fractions_from_state_kernel(int ns, int mode, int kind, int64_t n, int64_t tile,
                                                                   const double* __restrict__ wr, const double* __restrict__ phi,
                                                                   const double* __restrict__ param, double* __restrict__ frac) {
  const int64_t s = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (s >= n) return;
  const double* __restrict__ p = phi + conv_base(s, tile, ns + 1);
  double* __restrict__ f = frac + conv_base(s, tile, ns);
  const double T = p[0], E = p[tile], par = param[s];
  const double V = mode == PYJAC_CONP ? E : par, P = mode == PYJAC_CONP ? par : E;
  const double inv_ntot = R_GAS * T / (P * V);
  double sum = 0.0, wbar = 0.0;                           // sum of X_k and of X_k W_k / W_Ns over k < Ns
  for (int k = 0; k < ns - 1; ++k) { const double x = p[(int64_t)(2 + k) * tile] * inv_ntot; sum += x; wbar += x * __ldg(wr + k); }
  const double xl = 1.0 - sum;                            // the last species closes the ideal-gas law
  wbar += xl;                                             // wr[Ns-1] = 1
  const double iw = kind == PYJAC_MASS_FRACTION ? 1.0 / wbar : 1.0;
  for (int k = 0; k < ns - 1; ++k) {
    const double x = p[(int64_t)(2 + k) * tile] * inv_ntot;
    f[(int64_t)k * tile] = kind == PYJAC_MASS_FRACTION ? x * __ldg(wr + k) * iw : x;
  }
  f[(int64_t)(ns - 1) * tile] = xl * iw;
}
}  // namespace

struct pyjac_mech {
  int device = 0;
  int n_sm = 0;
  HostTables h;
  JacTables j;
  DevMech dm{};
  DevPlan plan[4]{};          // tile kernel (jacobian_kernel, pyjac_kernels.cu)
  DevPlan xplan[2]{};         // dense 'C' / 'F' by expansion (MODE 2): the sparse CSR / CSC plan + bitmap, ranks, scratch
  bool has_xplan = false;
  mutable cudaEvent_t scratch_ev = nullptr;   // launches that share the expansion scratch are ordered behind one another
  mutable bool scratch_used = false;
  DevJac dj{};                // pair kernel (jacobian2_kernel, pyjac_jacobian.cuh)
  DevJacOut jout[4]{};
  // pyjac_eval_host: two streams and two sets of staging buffers, created on first use and kept (grown when a call needs
  // more): the copy-inclusive path allocates nothing in steady state.  One eval_host call per handle at a time.
  struct HostStage {
    cudaStream_t st[2] = {nullptr, nullptr};
    double *phi[2] = {nullptr, nullptr}, *param[2] = {nullptr, nullptr}, *out[2] = {nullptr, nullptr};
    size_t phi_bytes = 0, param_bytes = 0, out_bytes = 0;
  };
  mutable HostStage stage;
  mutable std::mutex stage_mu;
  unsigned long long* static_sched = nullptr;   // device address of g_static_sched on this handle's device
  bool pair_only = false;     // the tile kernel's intermediates do not fit in shared memory, or PYJAC_PAIR_KERNEL
  std::vector<void*> allocs;
  // tile-scheduler words of the persistent Jacobian kernel: a ring of N_SCHED zeroed pairs (tile counter, finished
  // CTAs; the kernel leaves its pair zero again).  A launch takes the next pair; the event recorded behind the launch
  // that used the pair before tells whether that launch is still in flight (another stream), in which case the new
  // launch is ordered behind it: two kernels in flight never share a counter.
  static constexpr unsigned N_SCHED = 64;
  unsigned long long* sched = nullptr;
  mutable cudaEvent_t sched_ev[N_SCHED] = {};
  mutable bool sched_used[N_SCHED] = {};
  mutable unsigned sched_next = 0;
  mutable std::mutex sched_mu;
  ~pyjac_mech() {
    for (void* p : allocs) cudaFree(p);
    for (cudaEvent_t e : sched_ev) if (e) cudaEventDestroy(e);
    if (scratch_ev) cudaEventDestroy(scratch_ev);
    for (int b = 0; b < 2; ++b) {
      if (stage.st[b]) cudaStreamDestroy(stage.st[b]);
      cudaFree(stage.phi[b]); cudaFree(stage.param[b]); cudaFree(stage.out[b]);
    }
  }
  int upload_plan(const GatherPlan& g, int part_base, DevGather* out) {
    out->n_sg = g.n_sg; out->n_wide = g.n_wide; out->n_comb = (int)g.comb_item.size(); out->part_base = part_base;
    if (int r = upload(g.sg_meta, &out->sg_meta)) return r;
    if (int r = upload(g.comb_first, &out->comb_first)) return r;
    if (int r = upload(g.comb_nseg, &out->comb_nseg)) return r;
    return upload(g.ell_ent, &out->ell_ent);
  }
  template <class T> int upload(const std::vector<T>& v, const T** out) {
    void* p = nullptr;
    const size_t bytes = (v.size() ? v.size() : 1) * sizeof(T) + 32;   // +32: vector loads may touch padding
    CK(cudaMalloc(&p, bytes));
    allocs.push_back(p);
    CK(cudaMemset(p, 0, bytes));
    if (!v.empty()) CK(cudaMemcpy(p, v.data(), v.size() * sizeof(T), cudaMemcpyHostToDevice));
    *out = (const T*)p;
    return PYJAC_OK;
  }
};

extern "C" {

const char* pyjac_last_error(void) { return g_err.c_str(); }

int pyjac_mech_create(const pyjac_mech_desc* desc, int cuda_device, pyjac_mech** out) {
  return pyjac_mech_create_ex(desc, cuda_device, 0u, out);
}

int pyjac_mech_create_ex(const pyjac_mech_desc* desc, int cuda_device, uint32_t flags, pyjac_mech** out) {
  if (!desc || !out) return fail(PYJAC_EINVAL, "pyjac_mech_create: null argument");
  if (flags & ~(uint32_t)(PYJAC_APPROX_JACOBIAN | PYJAC_PAIR_KERNEL)) return fail(PYJAC_EINVAL, "pyjac_mech_create_ex: unknown flag");
  *out = nullptr;
  pyjac_mech* m = new (std::nothrow) pyjac_mech();
  if (!m) return fail(PYJAC_ENOMEM, "out of host memory");
  std::string err;
  int rc = build_host_tables(desc, (flags & PYJAC_APPROX_JACOBIAN) != 0, m->h, err);
  if (rc == PYJAC_OK) rc = build_jac_tables(m->h, m->j, err);
  // the tile kernel keeps ALL per-reaction partials of a state on chip; when they do not fit (or on request) the pair
  // kernel, which cuts the reactions into blocks, evaluates the Jacobian
  m->pair_only = (flags & PYJAC_PAIR_KERNEL) != 0 || choose_cfg(m->h, true, (int64_t)1 << 40, (int64_t)1 << 40, 148).smem > SMEM_LIMIT ||
                 !m->h.jplan.packable;    // (implied by the shared-memory test: 2^15 slots are 256 KB)
  if (rc != PYJAC_OK) { delete m; return fail(rc, err); }
  if (cuda_device == -1) { m->device = -1; *out = m; return PYJAC_OK; }   // host-only handle: pattern and dims only
  int ndev = 0;
  cudaError_t e = cudaGetDeviceCount(&ndev);
  if (e != cudaSuccess || cuda_device < 0 || cuda_device >= ndev) {
    delete m;
    return fail(PYJAC_ECUDA, "pyjac_mech_create: no CUDA device " + std::to_string(cuda_device) +
                                 (e != cudaSuccess ? std::string(" (") + cudaGetErrorString(e) + ")" : std::string()));
  }
  m->device = cuda_device;
  int prev = 0;
  cudaGetDevice(&prev);
  auto body = [&]() -> int {
    CK(cudaSetDevice(cuda_device));
    if (int ea = set_kernel_attributes()) return cuda_fail((cudaError_t)ea, "cudaFuncSetAttribute");
    if (int ea = set_kernel_attributes_jac()) return cuda_fail((cudaError_t)ea, "cudaFuncSetAttribute");
    CK(cudaDeviceGetAttribute(&m->n_sm, cudaDevAttrMultiProcessorCount, cuda_device));
    if (int rs_ = static_sched_address(cuda_device, &m->static_sched)) return rs_;
    for (unsigned q = 0; q < pyjac_mech::N_SCHED; ++q) CK(cudaEventCreateWithFlags(&m->sched_ev[q], cudaEventDisableTiming));
    {
      void* p = nullptr;
      CK(cudaMalloc(&p, pyjac_mech::N_SCHED * 2 * sizeof(unsigned long long)));
      m->allocs.push_back(p);
      CK(cudaMemset(p, 0, pyjac_mech::N_SCHED * 2 * sizeof(unsigned long long)));
      m->sched = (unsigned long long*)p;
    }
    HostTables& h = m->h;
    DevMech& d = m->dm;
    d.ns = h.ns; d.nr = h.nr; d.nvar = h.nvar; d.nslots = h.nslots;
    d.n_part_jac = h.n_part_jac; d.n_part_src = h.n_part_src;
#define UP(field) if (int r_ = m->upload(h.field, &d.field)) return r_;
    UP(nasa) UP(wr) UP(lnA) UP(beta) UP(Ta) UP(dn) UP(info) UP(aux) UP(sp) UP(eff_ptr) UP(eff_sp) UP(eff_d)
    UP(slot_base) UP(rev_par) UP(fall) UP(plog_ptr) UP(plog_ent) UP(plog_P) UP(plog_lnP) UP(plog_lnA) UP(plog_b) UP(plog_Ta)
    UP(cheb_meta) UP(cheb_lim) UP(cheb_coef)
#undef UP
    for (int ls = 0; ls < 6; ++ls) {
      if (int r_ = m->upload(h.rxc[ls], &d.rxc[ls])) return r_;
      d.n_rxc[ls] = (int)h.rxc[ls].size() / 2;
    }
    if (int r_ = m->upload_plan(h.cplan, h.jplan.n_part, &d.cplan)) return r_;      // C partials follow the J partials
    if (int r_ = m->upload_plan(h.qplan, 0, &d.qplan)) return r_;
    if (int r_ = m->upload(h.q_target, &d.q_target)) return r_;
    if (int r_ = m->upload(h.cplan.target, &d.c_item)) return r_;
    if (int r_ = m->upload(h.qplan.comb_item, &d.qc_item)) return r_;
    if (int r_ = m->upload(h.cplan.comb_item, &d.cc_item)) return r_;
    if (int r_ = m->upload(h.csc_ptr, &d.csc_ptr)) return r_;
    if (int r_ = m->upload(h.csc_idx, &d.csc_idx)) return r_;
    if (int r_ = m->upload(h.csc2csr, &d.csc2csr)) return r_;
    const uint32_t* mask[2];
    for (int p = 0; p < 2; ++p)
      if (int r_ = m->upload(h.nzmask[p], &mask[p])) return r_;
    {
      DevGather jplan;
      if (int r_ = m->upload_plan(h.jplan, 0, &jplan)) return r_;
      for (int f = 0; f < 4; ++f) {
        DevPlan& pl = m->plan[f];
        pl.n_e = f < 2 ? h.nnz : (int64_t)h.nvar * h.nvar;
        pl.jplan = jplan;
        if (int r_ = m->upload(h.j_pos[f], &pl.j_pos)) return r_;
        if (int r_ = m->upload(h.c_pos[f], &pl.c_pos)) return r_;
        if (int r_ = m->upload(h.jc_pos[f], &pl.jc_pos)) return r_;
        if (int r_ = m->upload(h.cc_pos[f], &pl.cc_pos)) return r_;
        for (int c = 0; c < 4; ++c) pl.d_pos[c] = h.d_pos[f][c];
        pl.nzmask = f < 2 ? nullptr : mask[f & 1];
        pl.xpair[0] = pl.xpair[1] = nullptr; pl.scratch = nullptr;
      }
      // dense by expansion: mechanisms that leave room for one state per CTA only, with a large dense matrix (C4)
      const bool one_state = choose_cfg(h, true, (int64_t)1 << 40, (int64_t)1 << 40, m->n_sm).S == 1;
      if (one_state && (int64_t)h.nvar * h.nvar >= 32768 && h.nnz < (1 << 29)) {
        void* scr = nullptr;
        CK(cudaMalloc(&scr, sizeof(double) * 2 * (size_t)m->n_sm * (size_t)h.nnz));   // two buffers (tile parity) per CTA
        m->allocs.push_back(scr);
        CK(cudaEventCreateWithFlags(&m->scratch_ev, cudaEventDisableTiming));
        for (int p = 0; p < 2; ++p) {
          DevPlan& x = m->xplan[p];
          x = m->plan[p];                          // positions of the CSR ('C') / CSC ('F') value order
          x.nzmask = mask[p];
          for (int sh = 0; sh < 2; ++sh)
            if (int r_ = m->upload(h.xpair[2 * p + sh], &x.xpair[sh])) return r_;
          x.scratch = (double*)scr;
        }
        m->has_xplan = true;
      }
    }
    // the pair kernel's own tables (block order) and plan
    {
      const JacTables& j = m->j;
      DevJac& q = m->dj;
      q.ns = j.ns; q.nr = j.nr; q.nvar = j.nvar; q.H = j.H; q.ns_max = j.ns_max; q.n_val = j.n_val; q.max_nrb = j.max_nrb;
      q.n_groups = (int)j.groups.size();
      for (int b = 0; b <= j.H; ++b) q.blk_r0[b] = j.blk_r0[b];
      for (int b = 0; b < j.H; ++b) q.blk_ng[b] = j.blk_ng[b];
      for (int b = 0; b <= j.H + 1; ++b) q.blk_g0[b] = j.blk_g0[b];
#define UPJ(field) if (int r_ = m->upload(j.field, &q.field)) return r_;
      UPJ(lnA) UPJ(beta) UPJ(Ta) UPJ(dn) UPJ(info) UPJ(sp) UPJ(ext) UPJ(groups) UPJ(ent) UPJ(pidx) UPJ(item) UPJ(nplus)
#undef UPJ
      q.nasa = d.nasa; q.eff_sp = d.eff_sp; q.eff_d = d.eff_d; q.rev_par = d.rev_par; q.fall = d.fall;
      q.plog_ptr = d.plog_ptr; q.plog_ent = d.plog_ent; q.plog_P = d.plog_P; q.plog_lnP = d.plog_lnP; q.plog_lnA = d.plog_lnA; q.plog_b = d.plog_b; q.plog_Ta = d.plog_Ta;
      q.cheb_meta = d.cheb_meta; q.cheb_lim = d.cheb_lim; q.cheb_coef = d.cheb_coef;
      for (int f = 0; f < 4; ++f) {
        DevJacOut& jo = m->jout[f];
        jo.n_e = f < 2 ? h.nnz : (int64_t)h.nvar * h.nvar;
        jo.pos16 = f < 2 && h.nnz < 65535;            // 16-bit output positions (0xffff = none)
        if (jo.pos16) {
          std::vector<uint16_t> a(j.posA[f].size()), b(j.posB[f].size());
          for (size_t e = 0; e < a.size(); ++e) { a[e] = (uint16_t)j.posA[f][e]; b[e] = (uint16_t)j.posB[f][e]; }   // J_NOPOS -> 0xffff
          const uint16_t *pa = nullptr, *pb = nullptr;
          if (int r_ = m->upload(a, &pa)) return r_;
          if (int r_ = m->upload(b, &pb)) return r_;
          jo.posA = pa; jo.posB = pb;
        } else {
          const uint32_t *pa = nullptr, *pb = nullptr;
          if (int r_ = m->upload(j.posA[f], &pa)) return r_;
          if (int r_ = m->upload(j.posB[f], &pb)) return r_;
          jo.posA = pa; jo.posB = pb;
        }
        for (int c = 0; c < 4; ++c) jo.d_pos[c] = j.d_pos[f][c];
        jo.nzmask = f < 2 ? nullptr : mask[f & 1];
      }
    }
    CK(cudaDeviceSynchronize());
    return PYJAC_OK;
  };
  rc = body();
  cudaSetDevice(prev);
  if (rc != PYJAC_OK) { delete m; return rc; }
  *out = m;
  return PYJAC_OK;
}

void pyjac_mech_destroy(pyjac_mech* mech) {
  if (!mech) return;
  if (mech->device < 0) { delete mech; return; }
  int prev = 0;
  cudaGetDevice(&prev);
  cudaSetDevice(mech->device);
  delete mech;
  cudaSetDevice(prev);
}

int pyjac_mech_dims(const pyjac_mech* mech, int32_t* ns, int32_t* nr, int32_t* nvar, int64_t* nnz) {
  if (!mech) return fail(PYJAC_EINVAL, "pyjac_mech_dims: null handle");
  if (ns) *ns = mech->h.ns;
  if (nr) *nr = mech->h.nr;
  if (nvar) *nvar = mech->h.nvar;
  if (nnz) *nnz = mech->h.nnz;
  return PYJAC_OK;
}

int pyjac_sparsity(const pyjac_mech* mech, int fmt, const int32_t** ptr, const int32_t** idx) {
  if (!mech || !ptr || !idx) return fail(PYJAC_EINVAL, "pyjac_sparsity: null argument");
  if (fmt != PYJAC_CSR && fmt != PYJAC_CSC) return fail(PYJAC_EINVAL, "pyjac_sparsity: fmt must be PYJAC_CSR or PYJAC_CSC");
  *ptr = fmt == PYJAC_CSR ? mech->h.csr_ptr.data() : mech->h.csc_ptr.data();
  *idx = fmt == PYJAC_CSR ? mech->h.csr_idx.data() : mech->h.csc_idx.data();
  return PYJAC_OK;
}

static int check_common(const char* fn, const pyjac_mech* mech, int mode, int64_t n_states, int64_t ld, int64_t tile,
                        const void* phi, const void* param, const void* out) {
  if (!mech) return fail(PYJAC_EINVAL, std::string(fn) + ": null handle");
  if (mech->device < 0) return fail(PYJAC_ECUDA, std::string(fn) + ": host-only handle (created with cuda_device = -1) cannot compute");
  if (mode != PYJAC_CONP && mode != PYJAC_CONV) return fail(PYJAC_EINVAL, std::string(fn) + ": mode must be PYJAC_CONP or PYJAC_CONV");
  if (n_states < 0) return fail(PYJAC_EINVAL, std::string(fn) + ": n_states < 0");
  if (ld < n_states) return fail(PYJAC_EINVAL, std::string(fn) + ": ld < n_states");
  if (tile < 1 || (tile != ld && (tile & (tile - 1)) != 0)) return fail(PYJAC_EINVAL, std::string(fn) + ": tile must be a power of two or equal to ld");
  if (n_states > 0 && ld % tile != 0) return fail(PYJAC_EINVAL, std::string(fn) + ": ld must be a multiple of tile");
  if (n_states > 0 && (!phi || !param || !out)) return fail(PYJAC_EINVAL, std::string(fn) + ": null buffer");
  if (((uintptr_t)phi | (uintptr_t)param | (uintptr_t)out) & 15) return fail(PYJAC_EINVAL, std::string(fn) + ": buffers must be 16-byte aligned");
  int cur = -1;
  if (cudaGetDevice(&cur) != cudaSuccess || cur != mech->device)
    return fail(PYJAC_EINVAL, std::string(fn) + ": the current CUDA device (" + std::to_string(cur) + ") is not the handle's device (" +
                                  std::to_string(mech->device) + ")");
  return PYJAC_OK;
}

int pyjac_source_terms(const pyjac_mech* mech, int mode, int64_t n_states, int64_t ld, int64_t tile, const double* d_phi,
                       const double* d_param, double* d_dphi, void* stream) {
  if (int rc = check_common("pyjac_source_terms", mech, mode, n_states, ld, tile, d_phi, d_param, d_dphi)) return rc;
  if (n_states == 0) return PYJAC_OK;
  const LaunchCfg cfg = choose_cfg(mech->h, false, tile, n_states, mech->n_sm);
  if (cfg.smem > SMEM_LIMIT) return fail(PYJAC_ENOMEM, "pyjac_source_terms: mechanism too large for shared memory");
  int e = launch_source(mech->dm, cfg, mode, n_states, ld, tile, d_phi, d_param, d_dphi, stream);
  if (e) return cuda_fail((cudaError_t)e, "source_kernel launch");
  return PYJAC_OK;
}

static int run_jac(const char* fn, const pyjac_mech* mech, int mode, int ofmt, int64_t n_states, int64_t ld, int64_t tile,
                   const double* d_phi, const double* d_param, double* d_out, void* stream) {
  if (int rc = check_common(fn, mech, mode, n_states, ld, tile, d_phi, d_param, d_out)) return rc;
  if (n_states == 0) return PYJAC_OK;
  const LaunchCfg cfg = mech->pair_only ? choose_cfg_jac(mech->j, tile, n_states, mech->n_sm) : choose_cfg(mech->h, true, tile, n_states, mech->n_sm);
  if (cfg.smem > J_SMEM_LIMIT) return fail(PYJAC_ENOMEM, std::string(fn) + ": mechanism too large for shared memory");
  std::lock_guard<std::mutex> lock(mech->sched_mu);
  const unsigned slot = mech->sched_next++ % pyjac_mech::N_SCHED;
  if (mech->sched_used[slot] && cudaEventQuery(mech->sched_ev[slot]) == cudaErrorNotReady)
    CK(cudaStreamWaitEvent((cudaStream_t)stream, mech->sched_ev[slot], 0));     // the pair's previous launch is still in flight
  (void)cudaGetLastError();                                                       // cudaErrorNotReady is not an error
  unsigned long long* sched = mech->sched + 2 * slot;
  // dense by expansion (one state per CTA, state-major layout): the launch uses the handle's scratch; it is ordered
  // behind the previous launch that did (another stream could still be running it)
  const bool expand = !mech->pair_only && mech->has_xplan && ofmt >= OUT_DENSE_C && cfg.S == 1 && tile == 1;
  if (expand && mech->scratch_used) CK(cudaStreamWaitEvent((cudaStream_t)stream, mech->scratch_ev, 0));
  const int e = mech->pair_only
                    ? launch_jacobian2(mech->dj, mech->jout[ofmt], cfg, mech->n_sm, mode, n_states, tile, d_phi, d_param, d_out, sched, stream)
                    : launch_jacobian(mech->dm, expand ? mech->xplan[ofmt - OUT_DENSE_C] : mech->plan[ofmt], cfg, mode, n_states, ld, tile, d_phi,
                                      d_param, d_out, sched, stream);
  if (e) return cuda_fail((cudaError_t)e, "jacobian kernel launch");
  if (expand) { CK(cudaEventRecord(mech->scratch_ev, (cudaStream_t)stream)); mech->scratch_used = true; }
  CK(cudaEventRecord(mech->sched_ev[slot], (cudaStream_t)stream));
  mech->sched_used[slot] = true;
  return PYJAC_OK;
}

int pyjac_jacobian_sparse(const pyjac_mech* mech, int mode, int fmt, int64_t n_states, int64_t ld, int64_t tile,
                          const double* d_phi, const double* d_param, double* d_vals, void* stream) {
  if (fmt != PYJAC_CSR && fmt != PYJAC_CSC) return fail(PYJAC_EINVAL, "pyjac_jacobian_sparse: fmt must be PYJAC_CSR or PYJAC_CSC");
  return run_jac("pyjac_jacobian_sparse", mech, mode, fmt == PYJAC_CSR ? OUT_CSR : OUT_CSC, n_states, ld, tile, d_phi, d_param, d_vals, stream);
}

int pyjac_jacobian_sparse_static(const pyjac_mech* mech, int mode, int fmt, int64_t n_states, int64_t ld, int64_t tile,
                                 const double* d_phi, const double* d_param, double* d_vals, void* stream) {
  const char* fn = "pyjac_jacobian_sparse_static";
  if (fmt != PYJAC_CSR && fmt != PYJAC_CSC) return fail(PYJAC_EINVAL, std::string(fn) + ": fmt must be PYJAC_CSR or PYJAC_CSC");
  if (int rc = check_common(fn, mech, mode, n_states, ld, tile, d_phi, d_param, d_vals)) return rc;
  if (n_states > PYJAC_STATIC_MAX_STATES)
    return fail(PYJAC_EINVAL, std::string(fn) + ": n_states " + std::to_string(n_states) + " exceeds PYJAC_STATIC_MAX_STATES = " +
                                  std::to_string((long long)PYJAC_STATIC_MAX_STATES) + " (split the batch, or use pyjac_jacobian_sparse)");
  if (n_states == 0) return PYJAC_OK;
  const LaunchCfg cfg = mech->pair_only ? choose_cfg_jac(mech->j, tile, n_states, mech->n_sm) : choose_cfg(mech->h, true, tile, n_states, mech->n_sm);
  if (cfg.smem > J_SMEM_LIMIT) return fail(PYJAC_ENOMEM, std::string(fn) + ": mechanism too large for shared memory");
  const int ofmt = fmt == PYJAC_CSR ? OUT_CSR : OUT_CSC;
  // every call shares the two words and they keep the last call's contents: they must start at zero (a launch that
  // faulted or was cancelled leaves them dirty), so they are cleared on the caller's stream in front of the kernel
  CK(cudaMemsetAsync(mech->static_sched, 0, 2 * sizeof(unsigned long long), (cudaStream_t)stream));
  const int e = mech->pair_only
                    ? launch_jacobian2(mech->dj, mech->jout[ofmt], cfg, mech->n_sm, mode, n_states, tile, d_phi, d_param, d_vals, mech->static_sched, stream)
                    : launch_jacobian(mech->dm, mech->plan[ofmt], cfg, mode, n_states, ld, tile, d_phi, d_param, d_vals, mech->static_sched, stream);
  if (e) return cuda_fail((cudaError_t)e, "jacobian kernel launch");
  return PYJAC_OK;
}

int pyjac_jacobian_dense(const pyjac_mech* mech, int mode, char order, int64_t n_states, int64_t ld, int64_t tile,
                         const double* d_phi, const double* d_param, double* d_J, void* stream) {
  if (order != 'C' && order != 'F') return fail(PYJAC_EINVAL, "pyjac_jacobian_dense: order must be 'C' or 'F'");
  return run_jac("pyjac_jacobian_dense", mech, mode, order == 'C' ? OUT_DENSE_C : OUT_DENSE_F, n_states, ld, tile, d_phi, d_param, d_J, stream);
}

int pyjac_jacobian_fd(const pyjac_mech* mech, int mode, int fmt, double rel_step, double abs_step, int64_t n_states,
                      int64_t ld, int64_t tile, const double* d_phi, const double* d_param, double* d_out, void* stream) {
  int ofmt;
  if (fmt == PYJAC_CSR) ofmt = OUT_CSR;
  else if (fmt == PYJAC_CSC) ofmt = OUT_CSC;
  else if (fmt == 'C') ofmt = OUT_DENSE_C;
  else if (fmt == 'F') ofmt = OUT_DENSE_F;
  else return fail(PYJAC_EINVAL, "pyjac_jacobian_fd: fmt must be PYJAC_CSR, PYJAC_CSC, 'C' or 'F'");
  if (!(rel_step >= 0.0) || !(abs_step >= 0.0) || !(rel_step + abs_step > 0.0))
    return fail(PYJAC_EINVAL, "pyjac_jacobian_fd: steps must be >= 0 and not both zero");
  if (int rc = check_common("pyjac_jacobian_fd", mech, mode, n_states, ld, tile, d_phi, d_param, d_out)) return rc;
  if (n_states == 0) return PYJAC_OK;
  const LaunchCfg cfg = choose_cfg_fd(mech->h);
  if (cfg.smem > SMEM_LIMIT) return fail(PYJAC_ENOMEM, "pyjac_jacobian_fd: mechanism too large for shared memory");
  const int64_t n_e = ofmt < OUT_DENSE_C ? mech->h.nnz : (int64_t)mech->h.nvar * mech->h.nvar;
  int e = launch_fd(mech->dm, cfg, mode, ofmt, n_e, rel_step, abs_step, n_states, ld, tile, d_phi, d_param, d_out, stream);
  if (e) return cuda_fail((cudaError_t)e, "fd_kernel launch");
  return PYJAC_OK;
}

int pyjac_launch_info(const pyjac_mech* mech, int what, int64_t n_states, int64_t tile, int32_t* states_per_cta, int32_t* threads,
                      int64_t* smem_bytes) {
  if (!mech) return fail(PYJAC_EINVAL, "pyjac_launch_info: null handle");
  if (what < 0 || what > 3) return fail(PYJAC_EINVAL, "pyjac_launch_info: what must be 0..3");
  if (n_states <= 0) n_states = (int64_t)1 << 40;          // "a large batch"
  if (tile <= 0) tile = (int64_t)1 << 40;                  // "any layout"
  const int n_sm = mech->n_sm > 0 ? mech->n_sm : 148;       // host-only handle: a B200's SM count, for reporting
  const LaunchCfg cfg = what == 3 ? choose_cfg_fd(mech->h)
                      : (what == 0 ? choose_cfg(mech->h, false, tile, n_states, n_sm)
                                   : (mech->pair_only ? choose_cfg_jac(mech->j, tile, n_states, n_sm) : choose_cfg(mech->h, true, tile, n_states, n_sm)));
  if (states_per_cta) *states_per_cta = cfg.S;
  if (threads) *threads = cfg.threads;
  if (smem_bytes) *smem_bytes = (int64_t)cfg.smem;
  return PYJAC_OK;
}

static int check_conv(const char* fn, const pyjac_mech* mech, int mode, int kind, int64_t n_states, int64_t ld, int64_t tile) {
  if (!mech) return fail(PYJAC_EINVAL, std::string(fn) + ": null handle");
  if (mech->device < 0) return fail(PYJAC_ECUDA, std::string(fn) + ": host-only handle (created with cuda_device = -1) cannot compute");
  if (mode != PYJAC_CONP && mode != PYJAC_CONV) return fail(PYJAC_EINVAL, std::string(fn) + ": mode must be PYJAC_CONP or PYJAC_CONV");
  if (kind != PYJAC_MOLE_FRACTION && kind != PYJAC_MASS_FRACTION) return fail(PYJAC_EINVAL, std::string(fn) + ": kind must be PYJAC_MOLE_FRACTION or PYJAC_MASS_FRACTION");
  if (n_states < 0 || ld < n_states) return fail(PYJAC_EINVAL, std::string(fn) + ": bad n_states / ld");
  if (tile < 1 || (tile != ld && (tile & (tile - 1)) != 0) || (n_states > 0 && ld % tile != 0))
    return fail(PYJAC_EINVAL, std::string(fn) + ": tile must be a power of two dividing ld, or equal to ld");
  return PYJAC_OK;
}

int pyjac_state_from_fractions(const pyjac_mech* mech, int mode, int kind, int64_t n_states, int64_t ld, int64_t tile,
                               const double* d_T, const double* d_P, const double* d_V, const double* d_frac, double* d_phi,
                               double* d_param, void* stream) {
  const char* fn = "pyjac_state_from_fractions";
  if (int rc = check_conv(fn, mech, mode, kind, n_states, ld, tile)) return rc;
  if (n_states == 0) return PYJAC_OK;
  if (!d_T || !d_P || !d_V || !d_frac || !d_phi || !d_param) return fail(PYJAC_EINVAL, std::string(fn) + ": null buffer");
  state_from_fractions_kernel<<<(unsigned)((n_states + 255) / 256), 256, 0, (cudaStream_t)stream>>>(
      mech->h.ns, mode, kind, n_states, tile, mech->dm.wr, d_T, d_P, d_V, d_frac, d_phi, d_param);
  CK(cudaGetLastError());
  return PYJAC_OK;
}

int pyjac_fractions_from_state(const pyjac_mech* mech, int mode, int kind, int64_t n_states, int64_t ld, int64_t tile,
                               const double* d_phi, const double* d_param, double* d_frac, void* stream) {
  const char* fn = "pyjac_fractions_from_state";
  if (int rc = check_conv(fn, mech, mode, kind, n_states, ld, tile)) return rc;
  if (n_states == 0) return PYJAC_OK;
  if (!d_phi || !d_param || !d_frac) return fail(PYJAC_EINVAL, std::string(fn) + ": null buffer");
  fractions_from_state_kernel<<<(unsigned)((n_states + 255) / 256), 256, 0, (cudaStream_t)stream>>>(
      mech->h.ns, mode, kind, n_states, tile, mech->dm.wr, d_phi, d_param, d_frac);
  CK(cudaGetLastError());
  return PYJAC_OK;
}

int pyjac_plan_info(const pyjac_mech* mech, int64_t info[8]) {
  if (!mech || !info) return fail(PYJAC_EINVAL, "pyjac_plan_info: null argument");
  const JacTables& j = mech->j;
  info[0] = j.H; info[1] = j.ns_max; info[2] = j.n_part; info[3] = j.n_entries; info[4] = j.n_padded;
  info[5] = (int64_t)j.groups.size(); info[6] = j.n_pieces; info[7] = j.n_span;
  return PYJAC_OK;
}

// copies `rows` rows of `n_c` states between a host array in the library layout (ld, tile) starting at state c0
// (c0 % tile == 0) and a device chunk buffer laid out with (ld = chunk, tile = tile_dev)
static cudaError_t copy_chunk(bool to_device, double* dev, const double* host_c, double* host, int64_t rows, int64_t c0,
                              int64_t n_c, int64_t ld, int64_t tile, int64_t chunk, int64_t tile_dev, cudaStream_t st) {
  const cudaMemcpyKind kind = to_device ? cudaMemcpyHostToDevice : cudaMemcpyDeviceToHost;
  if (tile == ld) {      // pure SoA: rows x n_c block of a rows x ld matrix; device chunk is rows x chunk
    if (to_device) return cudaMemcpy2DAsync(dev, chunk * 8, host_c + c0, ld * 8, n_c * 8, rows, kind, st);
    return cudaMemcpy2DAsync(host + c0, ld * 8, dev, chunk * 8, n_c * 8, rows, kind, st);
  }
  (void)tile_dev;        // == tile: whole tiles are contiguous runs of rows * tile doubles
  const int64_t full = n_c / tile, tail = n_c % tile;
  const int64_t hoff = (c0 / tile) * rows * tile;
  cudaError_t e = cudaSuccess;
  if (full) {
    if (to_device) e = cudaMemcpyAsync(dev, host_c + hoff, full * rows * tile * 8, kind, st);
    else e = cudaMemcpyAsync(host + hoff, dev, full * rows * tile * 8, kind, st);
    if (e != cudaSuccess) return e;
  }
  if (tail) {            // last partial tile: only the valid state slots (never touch s >= n_states)
    const int64_t o = full * rows * tile;
    if (to_device) e = cudaMemcpy2DAsync(dev + o, tile * 8, host_c + hoff + o, tile * 8, tail * 8, rows, kind, st);
    else e = cudaMemcpy2DAsync(host + hoff + o, tile * 8, dev + o, tile * 8, tail * 8, rows, kind, st);
  }
  return e;
}

int pyjac_eval_host(const pyjac_mech* mech, int what, int mode, int fmt, int64_t n_states, int64_t ld, int64_t tile,
                    const double* h_phi, const double* h_param, double* h_out) {
  if (!mech) return fail(PYJAC_EINVAL, "pyjac_eval_host: null handle");
  if (what < 0 || what > 2) return fail(PYJAC_EINVAL, "pyjac_eval_host: what must be 0, 1 or 2");
  if (n_states < 0 || ld < n_states) return fail(PYJAC_EINVAL, "pyjac_eval_host: bad n_states / ld");
  if (tile < 1 || (tile != ld && (tile & (tile - 1)) != 0) || (n_states > 0 && ld % tile != 0))
    return fail(PYJAC_EINVAL, "pyjac_eval_host: tile must be a power of two dividing ld, or equal to ld");
  if (mech->device < 0) return fail(PYJAC_ECUDA, "pyjac_eval_host: host-only handle cannot compute");
  if (n_states == 0) return PYJAC_OK;
  if (!h_phi || !h_param || !h_out) return fail(PYJAC_EINVAL, "pyjac_eval_host: null buffer");
  const int64_t nvar = mech->h.nvar;
  const int64_t n_e = what == 0 ? nvar : (what == 1 ? mech->h.nnz : nvar * nvar);
  // chunked, double-buffered pipeline: H2D(c+1) and D2H(c-1) overlap the kernel of chunk c when the host
  // buffers are pinned; with pageable memory the copies serialise but the result is the same
  int64_t chunk = 8192;
  while (chunk > 256 && chunk * n_e * 8 > (int64_t)1 << 30) chunk >>= 1;     // <= 1 GiB of output per buffer
  if (tile != ld && tile > chunk) chunk = tile;
  if (chunk > ld) chunk = ld;
  if (tile != ld) chunk -= chunk % tile;
  const int64_t tile_dev = tile == ld ? chunk : tile;
  int prev = 0;
  cudaGetDevice(&prev);
  std::lock_guard<std::mutex> stage_lock(mech->stage_mu);
  pyjac_mech::HostStage& sg = mech->stage;
  double **d_phi = sg.phi, **d_param = sg.param, **d_out = sg.out;
  cudaStream_t* st = sg.st;
  auto body = [&]() -> int {
    CK(cudaSetDevice(mech->device));
    auto grow = [&](double** buf, size_t& have, size_t need) -> int {
      if (need <= have) return PYJAC_OK;
      for (int b = 0; b < 2; ++b) { CK(cudaFree(buf[b])); buf[b] = nullptr; }
      have = 0;
      for (int b = 0; b < 2; ++b) CK(cudaMalloc(&buf[b], need));
      have = need;
      return PYJAC_OK;
    };
    for (int b = 0; b < 2; ++b)
      if (!st[b]) CK(cudaStreamCreateWithFlags(&st[b], cudaStreamNonBlocking));
    if (int rg = grow(d_phi, sg.phi_bytes, sizeof(double) * nvar * chunk)) return rg;
    if (int rg = grow(d_param, sg.param_bytes, sizeof(double) * chunk)) return rg;
    if (int rg = grow(d_out, sg.out_bytes, sizeof(double) * n_e * chunk)) return rg;
    int b = 0;
    for (int64_t c0 = 0; c0 < n_states; c0 += chunk, b ^= 1) {
      const int64_t n_c = n_states - c0 < chunk ? n_states - c0 : chunk;
      CK(copy_chunk(true, d_phi[b], h_phi, nullptr, nvar, c0, n_c, ld, tile, chunk, tile_dev, st[b]));
      CK(cudaMemcpyAsync(d_param[b], h_param + c0, n_c * 8, cudaMemcpyHostToDevice, st[b]));
      int rc;
      if (what == 0) rc = pyjac_source_terms(mech, mode, n_c, chunk, tile_dev, d_phi[b], d_param[b], d_out[b], st[b]);
      else if (what == 1) rc = pyjac_jacobian_sparse(mech, mode, fmt, n_c, chunk, tile_dev, d_phi[b], d_param[b], d_out[b], st[b]);
      else rc = pyjac_jacobian_dense(mech, mode, (char)fmt, n_c, chunk, tile_dev, d_phi[b], d_param[b], d_out[b], st[b]);
      if (rc) return rc;
      CK(copy_chunk(false, d_out[b], nullptr, h_out, n_e, c0, n_c, ld, tile, chunk, tile_dev, st[b]));
    }
    CK(cudaStreamSynchronize(st[0]));
    CK(cudaStreamSynchronize(st[1]));
    return PYJAC_OK;
  };
  int rc = body();
  for (int b = 0; b < 2; ++b)
    if (st[b]) cudaStreamSynchronize(st[b]);
  cudaSetDevice(prev);
  return rc;
}

}  // extern "C"
