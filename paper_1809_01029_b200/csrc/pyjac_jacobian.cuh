// Analytical Jacobian kernel for sm_100a (steps a1-a6, a8-a11 of SURVEY.md section 8a), fp64.
//
// A CTA owns a tile of S = 2 LS states and keeps every per-state intermediate on chip.  A THREAD OWNS ONE ITEM FOR A
// PAIR OF STATES: every value is a double2, so table words, plan entries, indices and addresses are decoded once per
// two states, shared memory is read with 16-byte loads and every nonzero leaves the SM as one 16-byte store.
//   phase 0  items = species         : concentrations (Eq. 6-7), NASA-7 thermo, D = sum C_k c_k
//   for every reaction block b (the reactions are cut into H blocks so that one block's partials fit, pyjac_plan.cpp):
//     phase 1  items = reactions     : k_f, K_c, k_r, third body / falloff, rates of progress and the per-reaction
//                                      partials dq_i/dT, dq_i/dE, dQ_i/dC_j -> value slots in shared memory
//     phase 2  items = list pieces   : every Jacobian nonzero gathers its static list of slots (plus entries, then minus
//                                      entries: no per-entry sign arithmetic); a list inside one block is finished in
//                                      registers and stored ONCE, a list that spans blocks carries a partial sum
//   final wave: lists with several segments per block are combined from their partial sums
// Replaces the paper's zero-fill + "J[idx] += ..." read-modify-write and its run-time index search
// (PAPER.md L345).  No tensor cores (nothing here is a dense contraction), no fast-math.
#pragma once
#include <cuda_runtime.h>

#include "pyjac_internal.h"
#include "pyjac_math.cuh"

namespace pyjac {
namespace jac2 {


constexpr int NT = J_NT, NW = J_NW;

struct D2 { double a, b; };
__device__ __forceinline__ D2 mk(double a, double b) { D2 r; r.a = a; r.b = b; return r; }
__device__ __forceinline__ D2 mk(double a) { return mk(a, a); }
__device__ __forceinline__ D2 operator+(D2 x, D2 y) { return mk(x.a + y.a, x.b + y.b); }
__device__ __forceinline__ D2 operator-(D2 x, D2 y) { return mk(x.a - y.a, x.b - y.b); }
__device__ __forceinline__ D2 operator*(D2 x, D2 y) { return mk(x.a * y.a, x.b * y.b); }
__device__ __forceinline__ D2 operator*(D2 x, double y) { return mk(x.a * y, x.b * y); }
__device__ __forceinline__ D2 operator*(double y, D2 x) { return mk(x.a * y, x.b * y); }
__device__ __forceinline__ D2 operator+(D2 x, double y) { return mk(x.a + y, x.b + y); }
__device__ __forceinline__ D2 operator-(D2 x, double y) { return mk(x.a - y, x.b - y); }
__device__ __forceinline__ D2 operator-(D2 x) { return mk(-x.a, -x.b); }
__device__ __forceinline__ D2& operator+=(D2& x, D2 y) { x.a += y.a; x.b += y.b; return x; }
__device__ __forceinline__ D2& operator-=(D2& x, D2 y) { x.a -= y.a; x.b -= y.b; return x; }
__device__ __forceinline__ D2 fma2(D2 x, D2 y, D2 z) { return mk(fma(x.a, y.a, z.a), fma(x.b, y.b, z.b)); }
__device__ __forceinline__ D2 fma2(double x, D2 y, D2 z) { return mk(fma(x, y.a, z.a), fma(x, y.b, z.b)); }
// The library exponential and logarithm are ~100 instructions each when inlined; the kernel's instruction working set has
// to fit the instruction caches (16 warps in different phases fetch different code), so every use shares one copy.
static __device__ __noinline__ double exp_lib(double x) { return exp(x); }
static __device__ __noinline__ double log_lib(double x) { return log(x); }
__device__ __forceinline__ D2 exp2_(D2 x) { return mk(exp_lib(x.a), exp_lib(x.b)); }
__device__ __forceinline__ D2 exp2_fast(D2 x) {
  D2 e = mk(exp_core(x.a), exp_core(x.b));
  if (!(exp_in_range(x.a) && exp_in_range(x.b))) e = exp2_(x);
  return e;
}
__device__ __forceinline__ D2 ld2(const D2* p) { const double2 v = *reinterpret_cast<const double2*>(p); return mk(v.x, v.y); }
__device__ __forceinline__ void st2(D2* p, D2 v) { *reinterpret_cast<double2*>(p) = make_double2(v.a, v.b); }
__device__ __forceinline__ D2 shfl_xor2(D2 v, int o) { return mk(__shfl_xor_sync(0xffffffffu, v.a, o), __shfl_xor_sync(0xffffffffu, v.b, o)); }

// Sums N per-lane values over the lanes that agree in their low log2(KEEP) bits by recursive halving: in every round
// with more than one value left a lane keeps half of its values and hands the other half to its partner, so 16 values
// cost 8 + 4 + 2 + 1 + 1 exchanges instead of 16 x 5.  store(j, sum) is called by exactly one lane per (j, low bits).
template <int N, int OFF, int KEEP>
struct WarpSum {
  template <class F>
  static __device__ __forceinline__ void run(double (&v)[N], int j0, bool owner, F store) {
    const int lane = threadIdx.x & 31;
    if constexpr (OFF < KEEP || OFF == 0) {
      if (owner) {
#pragma unroll
        for (int i = 0; i < N; ++i) store(j0 + i, v[i]);
      }
    } else if constexpr (N > 1) {
      const bool up = (lane & OFF) != 0;
      double h[N / 2];
#pragma unroll
      for (int i = 0; i < N / 2; ++i) {
        const double send = up ? v[i] : v[i + N / 2], keep = up ? v[i + N / 2] : v[i];
        h[i] = keep + __shfl_xor_sync(0xffffffffu, send, OFF);
      }
      WarpSum<N / 2, OFF / 2, KEEP>::run(h, j0 + (up ? N / 2 : 0), owner, store);
    } else {
      double h[1] = {v[0] + __shfl_xor_sync(0xffffffffu, v[0], OFF)};
      WarpSum<1, OFF / 2, KEEP>::run(h, j0, owner && !(lane & OFF), store);
    }
  }
};

// per-pair scalars in shared memory
enum { SC_T = 0, SC_V, SC_P, SC_INVT, SC_LNT, SC_CTOT, SC_RT, SC_LNP, SC_LNPRT, SC_EL, SC_CL, SC_DCL, SC_D, SC_DDDT, NSC_USED };
static_assert(NSC_USED <= J_NSC, "scalar area too small");

__device__ __forceinline__ int next_chunk(int* counter) {
  int c = 0;
  if ((threadIdx.x & 31) == 0) c = atomicAdd(counter, 1);
  return __shfl_sync(0xffffffffu, c, 0);
}

// element offset of (element 0, state s) in the library layout (s / tile) * (n_e * tile) + s % tile.  tile is a power of
// two (shift >= 0) or equal to ld (shift < 0: one tile holds every state), so no 64-bit division is needed.
__device__ __forceinline__ int64_t state_base(int64_t s, int shift, int64_t n_e) {
  return shift < 0 ? s : (((s >> shift) * n_e) << shift) + (s & (((int64_t)1 << shift) - 1));
}

__device__ __forceinline__ double ipow(double x, int n) {   // n in 0..3
  double r = 1.0;
  if (n >= 1) r = x;
  if (n >= 2) r *= x;
  if (n >= 3) r *= x;
  return r;
}
__device__ __forceinline__ double dpow(double x, int n) {   // n x^(n-1)
  return n == 0 ? 0.0 : (n == 1 ? 1.0 : (n == 2 ? 2.0 * x : 3.0 * x * x));
}

struct Blend { double F, dF_dPr, dF_dT; };
// Troe / SRI blending function and its partial derivatives (R2, R4-5)
static __device__ __noinline__ Blend blend(int type, bool hasT2, const double* __restrict__ fp, double T, double invT, double lnT, double Pr_in) {
  Blend b; b.F = 1.0; b.dF_dPr = 0.0; b.dF_dT = 0.0;
  const double LN10 = 2.302585092994045684, ILN10 = 0.434294481903251828;
  const double Pr = fmax(Pr_in, 1e-300);
  if (type == PYJAC_FALLOFF_TROE) {
    const double a = fp[4], iT3 = 1.0 / fp[5], iT1 = 1.0 / fp[6], T2 = fp[7];
    const double e3 = exp_lib(-T * iT3), e1 = exp_lib(-T * iT1);
    double Fc = (1.0 - a) * e3 + a * e1;
    double dFc = -(1.0 - a) * iT3 * e3 - a * iT1 * e1;
    if (hasT2) { const double e2 = exp_lib(-T2 * invT); Fc += e2; dFc += T2 * invT * invT * e2; }
    const double L = log_lib(Pr) * ILN10, Lc = log_lib(Fc) * ILN10;
    const double n = 0.75 - 1.27 * Lc;
    const double A = L - 0.4 - 0.67 * Lc;
    const double B = n - 0.14 * A;
    const double iB = 1.0 / B;
    const double f = A * iB;
    const double g = 1.0 / (1.0 + f * f);
    b.F = exp_lib(LN10 * Lc * g);
    const double dlogF_df = -2.0 * Lc * f * g * g;
    const double df_dL = n * iB * iB;
    const double df_dLc = (-0.67 * B + 1.1762 * A) * iB * iB;
    b.dF_dPr = b.F * dlogF_df * df_dL / Pr;
    b.dF_dT = b.F * (g + dlogF_df * df_dLc) * dFc / Fc;
  } else if (type == PYJAC_FALLOFF_SRI) {
    const double a = fp[4], bb = fp[5], ic = 1.0 / fp[6], d = fp[7], e = fp[8];
    const double L = log_lib(Pr) * ILN10;
    const double X = 1.0 / (1.0 + L * L);
    const double eb = exp_lib(-bb * invT), ec = exp_lib(-T * ic);
    const double base = a * eb + ec;
    const double dbase = a * bb * invT * invT * eb - ec * ic;
    const double lb = log_lib(base);
    b.F = d * exp_lib(X * lb + e * lnT);
    b.dF_dPr = b.F * lb * (-2.0 * L * X * X) * ILN10 / Pr;
    b.dF_dT = b.F * (X * dbase / base + e * invT);
  }
  return b;
}

// shared-memory carve-up (units of D2 unless noted); every per-pair array is [index][LS]
template <int LS>
struct Smem {
  D2 *sc, *C, *G, *Hh, *K, *dE, *V, *red;
  double* dn;
  int4* grp;
  __device__ __forceinline__ Smem(unsigned char* raw, const DevJac& m) {
    sc = reinterpret_cast<D2*>(raw);
    C = sc + 2 * J_NSC * LS; G = C + (m.ns + 1) * LS; Hh = G + (m.ns + 1) * LS; K = Hh + (m.ns + 1) * LS;
    dE = K + (m.ns + 1) * LS; V = dE + m.max_nrb * LS; red = V + m.n_val * LS;
    dn = reinterpret_cast<double*>(red + NW * J_NRED * LS);
    grp = reinterpret_cast<int4*>(dn + ((m.nr + 1) & ~1));
  }
};

// where this thread's pair of states lives in the output
struct Out {
  double *pa, *pb;     // element 0 of state a / b
  int64_t tile;
  bool full;           // both states valid and adjacent in memory (tile even): one 16-byte store
  bool va, vb;         // state valid (the slow path: ragged last pair, odd tile)
  __device__ __noinline__ void store_slow(uint32_t pos, double a, double b) const {
    const int64_t off = (int64_t)pos * tile;
    if (va) __stcs(pa + off, a);
    if (vb) __stcs(pb + off, b);
  }
  __device__ __forceinline__ void store(uint32_t pos, D2 v) const {
    if (full) __stcs(reinterpret_cast<double2*>(pa + (int64_t)pos * tile), make_double2(v.a, v.b));
    else store_slow(pos, v.a, v.b);
  }
};

template <class PosT> __device__ __forceinline__ bool has_pos(PosT p) { return p != (PosT)~(PosT)0; }

// ---------------------------------------------------------------------------------------------------
// phase 2: the gather engine.  A unit = U x (32 / LS) pieces of one group; a thread owns U pieces (U independent
// chains of loads per step) for its pair of states.
// ---------------------------------------------------------------------------------------------------
template <int LS, class PosT>
__device__ __forceinline__ void gather_unit(const DevJac& m, const DevJacOut& o, const Smem<LS>& sm, const JGroup g, int sub,
                                            const Out& out, bool conp, int blk_r0) {
  constexpr int IPW = 32 / LS, U = 4, R = 1, RR = 1;   // pair steps requested at once: R (one word per step), RR (JK_ROW: two)
  const int lane = threadIdx.x & 31, pr = lane % LS, il = lane / LS;
  const D2* __restrict__ V = sm.V + pr;
  const PosT* __restrict__ posA = reinterpret_cast<const PosT*>(o.posA) + g.piece_off;
  const PosT* __restrict__ posB = reinterpret_cast<const PosT*>(o.posB) + g.piece_off;
  const uint16_t* __restrict__ pidx = m.pidx + g.piece_off;
  const uint8_t* __restrict__ nplus = m.nplus + g.piece_off;
  const int cls = g.cls;
  if (g.kind == JK_BLK1) {
    // lists of exactly one entry: J_GW1 pieces per group, 2 U per thread and unit
    constexpr int U1 = 2 * U;
    const int p0 = sub * (U1 * IPW) + il;
    const uint16_t* __restrict__ e = reinterpret_cast<const uint16_t*>(m.ent + g.ent_off) + p0;
    uint32_t idx[U1]; PosT pos[U1];
#pragma unroll
    for (int u = 0; u < U1; ++u) { idx[u] = __ldg(e + u * IPW); pos[u] = __ldg(posA + p0 + u * IPW); }
    const bool minus = g.nM2 != 0;
#pragma unroll
    for (int u = 0; u < U1; ++u) {
      D2 v = ld2(V + idx[u] * LS);
      if (minus) v = -v;
      if (has_pos(pos[u])) out.store(pos[u], v);
    }
    return;
  }
  const int p0 = sub * (U * IPW) + il;
  const int nP2 = g.nP2, nM2 = g.nM2;
  // pair steps needed by the quarter of the group that this thread's u-th piece belongs to (warp-uniform, descending)
  int nb[U];
#pragma unroll
  for (int u = 0; u < U; ++u) nb[u] = (int)((g.qsteps >> (8 * ((sub * U + u) / LS))) & 0xffu);
  (void)nP2;
  if (g.kind == JK_BLK) {
    const uint32_t* __restrict__ e = m.ent + g.ent_off + p0;
    PosT pos[U]; uint32_t pi[U];
#pragma unroll
    for (int u = 0; u < U; ++u) {
      pos[u] = (cls == JC_OUT || cls == JC_LAST) ? __ldg(posA + p0 + u * IPW) : (PosT)0;
      pi[u] = cls != JC_OUT ? __ldg(pidx + p0 + u * IPW) : 0u;
    }
    D2 v[U];
    int np[U];
#pragma unroll
    for (int u = 0; u < U; ++u) { v[u] = mk(0.0); np[u] = __ldg(nplus + p0 + u * IPW); }
    // entries 2 s and 2 s + 1 of a piece have one sign: plus while s < nplus, then minus (a multiplier of +-1 in the
    // DFMA: no sign arithmetic on the values)
    // rounds of R pair steps: every entry word of a round is requested before the first one is used (one exposed L2
    // round trip per round instead of one per step: the gathers are latency bound)
#pragma unroll 1
    for (int s0 = 0; s0 < nb[0]; s0 += R) {
      uint32_t w[R][U];
#pragma unroll
      for (int q = 0; q < R; ++q)
#pragma unroll
        for (int u = 0; u < U; ++u) w[q][u] = s0 + q < nb[u] ? __ldg(e + (s0 + q) * J_GW + u * IPW) : 0u;
#pragma unroll
      for (int q = 0; q < R; ++q)
#pragma unroll
        for (int u = 0; u < U; ++u) {
          if (s0 + q < nb[u]) {
            const double sg = s0 + q < np[u] ? 1.0 : -1.0;
            v[u] = fma2(sg, ld2(V + (w[q][u] & 0xffffu) * LS), v[u]);
            v[u] = fma2(sg, ld2(V + (w[q][u] >> 16) * LS), v[u]);
          }
        }
    }
#pragma unroll
    for (int u = 0; u < U; ++u) {
      D2* part = sm.V + pi[u] * LS + pr;
      if (cls == JC_OUT) { if (has_pos(pos[u])) out.store(pos[u], v[u]); }
      else if (cls == JC_FIRST) st2(part, v[u]);
      else if (cls == JC_ADD) st2(part, ld2(part) + v[u]);
      else if (has_pos(pos[u])) out.store(pos[u], v[u] + ld2(part));
    }
    return;
  }
  // two sums per piece
  PosT pa[U], pb[U]; uint32_t pi[U], it[U];
#pragma unroll
  for (int u = 0; u < U; ++u) {
    const bool fin = cls == JC_OUT || cls == JC_LAST;
    pa[u] = fin ? __ldg(posA + p0 + u * IPW) : (PosT)0;
    pb[u] = fin ? __ldg(posB + p0 + u * IPW) : (PosT)0;
    pi[u] = cls != JC_OUT ? __ldg(pidx + p0 + u * IPW) : 0u;
    it[u] = fin && g.kind != JK_COL ? __ldg(m.item + g.piece_off + p0 + u * IPW) : 0u;
  }
  D2 v0[U], v1[U];
#pragma unroll
  for (int u = 0; u < U; ++u) { v0[u] = mk(0.0); v1[u] = mk(0.0); }
  if (g.kind == JK_ROW) {
    // J[T][j] ~ sum_i dE~_i g_ij, J[E][j] ~ sum_i dn~_i g_ij: entry = slot | reaction-in-block << 16
    const uint2* __restrict__ e = reinterpret_cast<const uint2*>(m.ent + g.ent_off) + p0;
    const D2* __restrict__ dE = sm.dE + pr;
    const double* __restrict__ dn = sm.dn + blk_r0;
    auto acc = [&](uint32_t w, int u, bool minus) {
      const D2 x = ld2(V + (w & 0xffffu) * LS);
      const D2 de = ld2(dE + (w >> 16) * LS);
      const double d = dn[w >> 16];
      if (!minus) { v0[u] = fma2(de, x, v0[u]); v1[u] = fma2(d, x, v1[u]); }
      else { v0[u] = fma2(-de, x, v0[u]); v1[u] = fma2(-d, x, v1[u]); }
    };
#pragma unroll 1
    for (int s0 = 0; s0 < nb[0]; s0 += RR) {
      uint2 w[RR][U];
#pragma unroll
      for (int q = 0; q < RR; ++q)
#pragma unroll
        for (int u = 0; u < U; ++u) w[q][u] = s0 + q < nb[u] ? __ldg(e + (s0 + q) * J_GW + u * IPW) : make_uint2(0u, 0u);
#pragma unroll
      for (int q = 0; q < RR; ++q)
#pragma unroll
        for (int u = 0; u < U; ++u) if (s0 + q < nb[u]) { acc(w[q][u].x, u, false); acc(w[q][u].y, u, false); }
    }
    e += nP2 * J_GW;
    for (int s = 0; s < nM2; ++s) {
      uint2 w[U];
#pragma unroll
      for (int u = 0; u < U; ++u) w[u] = __ldg(e + s * J_GW + u * IPW);
#pragma unroll
      for (int u = 0; u < U; ++u) { acc(w[u].x, u, true); acc(w[u].y, u, true); }
    }
  } else {
    // JK_COL: J[k][T] = sum_i nu_ki slotT_i, J[k][E] = sum_i nu_ki slotE_i (slot E = slot T + 8); JK_ROWC: partial sums
    const uint32_t* __restrict__ e = m.ent + g.ent_off + p0;
    const D2* __restrict__ V8 = V + 8 * LS;
    int np[U];
#pragma unroll
    for (int u = 0; u < U; ++u) np[u] = __ldg(nplus + p0 + u * IPW);
#pragma unroll 1
    for (int s0 = 0; s0 < nb[0]; s0 += R) {
      uint32_t w[R][U];
#pragma unroll
      for (int q = 0; q < R; ++q)
#pragma unroll
        for (int u = 0; u < U; ++u) w[q][u] = s0 + q < nb[u] ? __ldg(e + (s0 + q) * J_GW + u * IPW) : 0u;
#pragma unroll
      for (int q = 0; q < R; ++q)
#pragma unroll
        for (int u = 0; u < U; ++u) {
          if (s0 + q < nb[u]) {
            const uint32_t i0 = (w[q][u] & 0xffffu) * LS, i1 = (w[q][u] >> 16) * LS;
            const double sg = s0 + q < np[u] ? 1.0 : -1.0;
            v0[u] = fma2(sg, ld2(V + i0), v0[u]); v1[u] = fma2(sg, ld2(V8 + i0), v1[u]);
            v0[u] = fma2(sg, ld2(V + i1), v0[u]); v1[u] = fma2(sg, ld2(V8 + i1), v1[u]);
          }
        }
    }
  }
  // factors of the T / E rows (only units that finish such rows get here with kind != JK_COL: a few per tile)
  D2 fT = mk(0.0), iDV = mk(0.0), cS = mk(0.0), cT = mk(0.0), cL = mk(0.0);
  if (g.kind != JK_COL && (cls == JC_OUT || cls == JC_LAST)) {
    D2 N = mk(0.0);
    for (int w = 0; w < NW; ++w) N += ld2(sm.red + (w * J_NRED + 0) * LS + pr);
    const D2 D = ld2(sm.sc + SC_D * LS + pr), T = ld2(sm.sc + SC_T * LS + pr), V_ = ld2(sm.sc + SC_V * LS + pr), Pp = ld2(sm.sc + SC_P * LS + pr);
    fT = mk(-N.a / D.a, -N.b / D.b);
    iDV = mk(1.0 / (D.a * V_.a), 1.0 / (D.b * V_.b));
    cS = conp ? mk(T.a * R_GAS / Pp.a, T.b * R_GAS / Pp.b) : mk(T.a * R_GAS / V_.a, T.b * R_GAS / V_.b);
    cT = conp ? mk(V_.a / T.a, V_.b / T.b) : mk(Pp.a / T.a, Pp.b / T.b);
    cL = ld2(sm.sc + SC_CL * LS + pr);
  }
#pragma unroll
  for (int u = 0; u < U; ++u) {
    D2* part = sm.V + pi[u] * LS + pr;
    if (cls == JC_FIRST) { st2(part, v0[u]); st2(part + 8 * LS, v1[u]); continue; }
    if (cls == JC_ADD) { st2(part, ld2(part) + v0[u]); st2(part + 8 * LS, ld2(part + 8 * LS) + v1[u]); continue; }
    if (cls == JC_LAST) { v0[u] += ld2(part); v1[u] += ld2(part + 8 * LS); }
    if (!has_pos(pa[u])) continue;
    if (g.kind == JK_COL) { out.store(pa[u], v0[u]); out.store(pb[u], v1[u]); }
    else {
      // a10: J[T][j] = -(sum_i dE~_i g_ij + f_T (c_j - c_Ns)) / (D V);  J[E][j] = cS sum_i dn~_i g_ij + cT J[T][j]
      const D2 cj = ld2(sm.K + it[u] * LS + pr);
      const D2 JT = -((v0[u] + fT * (cj - cL)) * iDV);
      out.store(pa[u], JT);
      out.store(pb[u], cS * v1[u] + cT * JT);
    }
  }
}

// ---------------------------------------------------------------------------------------------------
// phase 1, general path (any reaction type, any coefficients, the last species in any role): one STATE at a time,
// scalar code.  Shared arrays are addressed as doubles: element (i, pair, st) at ((i * LS + pr) * 2 + st).
// Returns the reaction's contributions to the seven reaction sums in inc[].
// ---------------------------------------------------------------------------------------------------
template <int LS>
__device__ __forceinline__ void reaction_general(const DevJac& m, const Smem<LS>& sm, int r, int lr, int pr, int st, bool conp,
                                              uint32_t info, uint4 spw, double (&inc)[7]) {
  const int ns = m.ns, L = ns - 1;
  const double* __restrict__ scd = reinterpret_cast<const double*>(sm.sc);
  auto sc = [&](int i) { return scd[(i * LS + pr) * 2 + st]; };
  auto sp_arr = [&](const D2* a, int k) { return reinterpret_cast<const double*>(a)[(k * LS + pr) * 2 + st]; };
  const double T = sc(SC_T), V = sc(SC_V), Pp = sc(SC_P), invT = sc(SC_INVT), lnT = sc(SC_LNT), Ctot = sc(SC_CTOT), RT = sc(SC_RT);
  const double lnP = sc(SC_LNP), ln_patm_rt = sc(SC_LNPRT), eL = sc(SC_EL), cL = sc(SC_CL);
  const double ctot_T = Ctot * invT;
  const int type = info & JI_TYPE_MASK;
  const bool rev = info & JI_REV;
  const int4 ext = __ldg(reinterpret_cast<const int4*>(m.ext) + r);
  const int rx_aux = ext.x, e0 = ext.y, e1 = ext.y + ext.z;
  const double rx_lnA = __ldg(m.lnA + r), rx_beta = __ldg(m.beta + r), rx_Ta = __ldg(m.Ta + r), dn = sm.dn[r];
  // a3: forward rate constant
  double lnkf, lam_f, dlnk_dP = 0.0;
  if (type <= PYJAC_FALLOFF_SRI) {
    lnkf = rx_lnA + rx_beta * lnT - rx_Ta * invT;
    lam_f = (rx_beta + rx_Ta * invT) * invT;
  } else if (type == PYJAC_PLOG) {
    const int p0 = __ldg(m.plog_ptr + rx_aux), np = __ldg(m.plog_ptr + rx_aux + 1) - p0;
    int cnt_le = 0;                                   // number of table pressures <= P
    for (int q = 0; q < np; ++q) cnt_le += __ldg(m.plog_P + p0 + q) <= Pp ? 1 : 0;
    // P <= P_0: first point; P >= P_last: last point; else interval j = last j with P_j <= P (S4)
    const bool interp = cnt_le >= 1 && cnt_le < np && !(cnt_le == 1 && Pp <= __ldg(m.plog_P + p0));
    const int j = cnt_le >= np ? np - 1 : (cnt_le >= 1 ? cnt_le - 1 : 0);
    const int j1 = interp ? j + 1 : j;
    // a pressure level is one entry, or several entries of equal pressure whose rates are summed (R10)
    auto level = [&](int l, double& lnk, double& lam) {
      const int q0 = __ldg(m.plog_ent + p0 + l), q1 = __ldg(m.plog_ent + p0 + l + 1);
      const double bq = __ldg(m.plog_b + q0), Taq = __ldg(m.plog_Ta + q0), lAq = __ldg(m.plog_lnA + q0);
      lnk = lAq + bq * lnT - Taq * invT;
      lam = (bq + Taq * invT) * invT;
      if (q1 - q0 > 1) {
        double ksum = exp_lib(lnk), dsum = ksum * lam;
        for (int e = q0 + 1; e < q1; ++e) {
          const double be = __ldg(m.plog_b + e), Tae = __ldg(m.plog_Ta + e);
          const double ke = exp_lib(__ldg(m.plog_lnA + e) + be * lnT - Tae * invT);
          ksum += ke; dsum += ke * ((be + Tae * invT) * invT);
        }
        lnk = log_lib(ksum); lam = dsum / ksum;
      }
    };
    const double lP0 = __ldg(m.plog_lnP + p0 + j), lP1 = __ldg(m.plog_lnP + p0 + j1);
    double l0, lam0, l1 = 0.0, lam1 = 0.0;
    level(j, l0, lam0);
    if (interp) level(j1, l1, lam1);
    lnkf = l0; lam_f = lam0;
    if (interp) {
      const double idl = 1.0 / (lP1 - lP0);
      const double w = (lnP - lP0) * idl;
      lnkf = l0 + (l1 - l0) * w;
      lam_f = (1.0 - w) * lam0 + w * lam1;
      dlnk_dP = (l1 - l0) * idl / Pp;
    }
  } else {
    const double LN10 = 2.302585092994045684, ILN10 = 0.434294481903251828;
    const int4 cm = __ldg(reinterpret_cast<const int4*>(m.cheb_meta) + rx_aux);          // nT, nP, coefficient offset
    const double2 cl0 = __ldg(reinterpret_cast<const double2*>(m.cheb_lim) + 2 * rx_aux);
    const double2 cl1 = __ldg(reinterpret_cast<const double2*>(m.cheb_lim) + 2 * rx_aux + 1);
    const int nP = cm.y, n_coef = cm.x * cm.y;
    const double* __restrict__ eta = m.cheb_coef + cm.z;
    const double iTmin = cl0.x, iTmax = cl0.y, lPmin = cl1.x, lPmax = cl1.y;
    const double Tr = (2.0 * invT - iTmin - iTmax) / (iTmax - iTmin);
    const double Pr_ = (2.0 * lnP * ILN10 - lPmin - lPmax) / (lPmax - lPmin);
    double lg = 0.0, dlg_dT = 0.0, dlg_dP = 0.0;
    // the row-major coefficients are consumed in order by a running pair of three-term recurrences
    double cT = 1.0, cTm = 0.0, dT = 0.0, dTm = 0.0;       // T_a(Tr), T_{a-1}, derivatives
    double cP = 1.0, cPm = 0.0, dP = 0.0, dPm = 0.0;
    int ia = 0, ib = 0;
    for (int q = 0; q < n_coef; ++q) {
      const double e = __ldg(eta + q);
      lg += e * cT * cP; dlg_dT += e * dT * cP; dlg_dP += e * cT * dP;
      if (++ib == nP) {                    // next row: advance T_a, restart T_b
        ib = 0; ++ia;
        if (ia == 1) { cTm = 1.0; cT = Tr; dTm = 0.0; dT = 1.0; }
        else { const double n1 = 2.0 * Tr * cT - cTm, d1 = 2.0 * cT + 2.0 * Tr * dT - dTm; cTm = cT; cT = n1; dTm = dT; dT = d1; }
        cP = 1.0; cPm = 0.0; dP = 0.0; dPm = 0.0;
      } else if (ib == 1) { cPm = 1.0; cP = Pr_; dPm = 0.0; dP = 1.0; }
      else { const double n1 = 2.0 * Pr_ * cP - cPm, d1 = 2.0 * cP + 2.0 * Pr_ * dP - dPm; cPm = cP; cP = n1; dPm = dP; dP = d1; }
    }
    lnkf = LN10 * lg;
    lam_f = LN10 * dlg_dT * (-2.0 * invT * invT / (iTmax - iTmin));
    dlnk_dP = dlg_dP * 2.0 / (Pp * (lPmax - lPmin));
  }
  const double kf = exp_lib(lnkf);
  // stoichiometry: concentrations, powers and one-factor-removed products (no division by C_k: DESIGN.md S7).
  // Unused entries point at the dummy species ns (C = 1, thermo = 0).
  const uint32_t spk[6] = {spw.x & 0xffffu, spw.x >> 16, spw.y & 0xffffu, spw.y >> 16, spw.z & 0xffffu, spw.z >> 16};
  const uint32_t nu_bits = spw.w >> 16;
  double pw[6], pm[6];
  double dg = 0.0, dh = 0.0, dc = 0.0;
#pragma unroll
  for (int a = 0; a < 6; ++a) {
    const int k = (int)spk[a], nu = (int)((nu_bits >> (2 * a)) & 3u);
    const double Ck = sp_arr(sm.C, k);
    pw[a] = ipow(Ck, nu); pm[a] = dpow(Ck, nu);
    const double snu = a < 3 ? -(double)nu : (double)nu;
    dg += snu * sp_arr(sm.G, k); dh += snu * sp_arr(sm.Hh, k); dc += snu * sp_arr(sm.K, k);
  }
  const double Pif = pw[0] * pw[1] * pw[2], Pir = pw[3] * pw[4] * pw[5];
  const double snu = (double)((int)((info >> JI_SNU_SHIFT) & 31u) - 16);
  double kr = 0.0, lam_r = 0.0;
  if (rev) {      // a4: K_c from Gibbs polynomials; k_r = k_f / K_c = exp_lib(ln k_f - ln K_c)
    if (info & JI_REVX) {        // explicit reverse Arrhenius parameters (R9): K_c plays no role
      const int ro = ext.w;
      const double lAr = __ldg(m.rev_par + 3 * ro), br = __ldg(m.rev_par + 3 * ro + 1), Tar = __ldg(m.rev_par + 3 * ro + 2);
      kr = exp_lib(lAr + br * lnT - Tar * invT);
      lam_r = (br + Tar * invT) * invT;
    } else {
      kr = exp_lib(lnkf + dg - snu * ln_patm_rt);
      lam_r = lam_f - (dh - snu) * invT;
    }
  }
  const double Rf = kf * Pif, Rr = kr * Pir, Rn = Rf - Rr;
  const double dRdT = lam_f * Rf - lam_r * Rr;
  // a5: third body / falloff
  double c = 1.0, X = 0.0, GT = dRdT, MdcdM_R = 0.0;
  const double adef = (info & JI_ADEF) ? 1.0 : 0.0;
  if (type >= PYJAC_THIRD_BODY && type <= PYJAC_FALLOFF_SRI) {
    double M = adef * Ctot;                       // sum_k C_k == C_tot by construction of C_Ns
    for (int eb = e0; eb < e1; ++eb) M += __ldg(m.eff_d + eb) * sp_arr(sm.C, __ldg(m.eff_sp + eb));
    if (type == PYJAC_THIRD_BODY) {
      c = M; X = Rn; GT = M * dRdT; MdcdM_R = M * Rn;
    } else {
      double fp[10];
      {
        const double2* __restrict__ f2 = reinterpret_cast<const double2*>(m.fall + 12 * rx_aux);
#pragma unroll
        for (int q = 0; q < 5; ++q) { const double2 v2 = __ldg(f2 + q); fp[2 * q] = v2.x; fp[2 * q + 1] = v2.y; }
      }
      // falloff: the record holds k_0 and lnkf = ln k_inf.  Chemically activated (R8): the record holds k_inf and
      // lnkf = ln k_0, so the ratio k_0 / k_inf and its temperature derivative change sign in the exponent, and
      // c = F / (1 + Pr) instead of F Pr / (1 + Pr).
      const bool chem = (info & JI_CHEM) != 0;
      const double b0 = fp[1], Ta0 = fp[2];
      const double lnrat = fp[0] + b0 * lnT - Ta0 * invT - lnkf;
      const double k0_kinf = exp_lib(chem ? -lnrat : lnrat);
      const double Pr = k0_kinf * M;
      const Blend bl = blend(type, info & JI_T2, fp, T, invT, lnT, Pr);
      const double i1p = 1.0 / (1.0 + Pr);
      const double cF = chem ? i1p : Pr * i1p;            // dc/dF
      c = bl.F * cF;
      const double dc_dPr = (chem ? -bl.F : bl.F) * i1p * i1p + cF * bl.dF_dPr;
      const double dlnrat_dT = (b0 - rx_beta + (Ta0 - rx_Ta) * invT) * invT;
      const double dPr_dT = Pr * (chem ? -dlnrat_dT : dlnrat_dT);
      X = dc_dPr * k0_kinf * Rn;
      GT = (dc_dPr * dPr_dT + cF * bl.dF_dT) * Rn + c * dRdT;
      MdcdM_R = Pr * dc_dPr * Rn;
    }
  }
  const double q = c * Rn;
  // reaction sums (R4-7/8): dE~_i = sum_k nu_ki (E_k - w_k E_Ns) = RT (sum nu_k e_k - e_Ns sum nu_k w_k) with
  // sum_k nu_ki w_k = sum(nu) - dn~_i; likewise dc~_i
  const double conv = conp ? 0.0 : 1.0;
  const double dEt = RT * (dh - conv * snu - eL * (snu - dn));
  const double dct = dc - cL * (snu - dn);
  // a8: per-reaction partials -> value slots (slot i at base + 8 i)
  double* __restrict__ Vd = reinterpret_cast<double*>(sm.V);
  const int sbase = (int)(spw.w & 0xffffu);
  auto slot = [&](int i) -> double& { return Vd[((sbase + 8 * i) * LS + pr) * 2 + st]; };
  const int nre = (info >> JI_NREAC_SHIFT) & 3, npr = (info >> JI_NPROD_SHIFT) & 3;
  const double a_ = c * kf, b_ = c * kr;
  double GL = adef * X;                          // full dQ_i/dC_Ns
  const double df[3] = {a_ * pm[0] * pw[1] * pw[2], a_ * pw[0] * pm[1] * pw[2], a_ * pw[0] * pw[1] * pm[2]};
  const double dr[3] = {-b_ * pm[3] * pw[4] * pw[5], -b_ * pw[3] * pm[4] * pw[5], -b_ * pw[3] * pw[4] * pm[5]};
  int si = 2;
#pragma unroll
  for (int a = 0; a < 3; ++a)
    if (a < nre) { slot(si++) = df[a]; if ((int)spk[a] == L) GL += df[a]; }
  if (rev) {
#pragma unroll
    for (int a = 0; a < 3; ++a)
      if (a < npr) { slot(si++) = dr[a]; if ((int)spk[3 + a] == L) GL += dr[a]; }
  }
  for (int eb = e0; eb < e1; ++eb) {
    const double v = __ldg(m.eff_d + eb) * X;
    slot(si++) = v;
    if (__ldg(m.eff_sp + eb) == L) GL += v;
  }
  // chain rule to the state variables (R4-2); E column in Euler-homogeneity form (R4-6)
  const double slotT = V * (GT - ctot_T * GL);
  double slotE;
  if (conp) {
    const int of = (info >> JI_OF_SHIFT) & 15, orv = (info >> JI_OR_SHIFT) & 15;
    slotE = q - c * ((double)of * Rf - (double)orv * Rr) - MdcdM_R + Ctot * GL;
  } else {
    slotE = V * (c * dlnk_dP * Rn + GL / RT);
  }
  slot(0) = slotT;
  slot(1) = slotE;
  reinterpret_cast<double*>(sm.dE)[(lr * LS + pr) * 2 + st] = dEt;
  inc[0] = dEt * q; inc[1] = dn * q; inc[2] = dEt * slotT; inc[3] = dn * slotT; inc[4] = dEt * slotE; inc[5] = dn * slotE; inc[6] = dct * q;
}

// ---------------------------------------------------------------------------------------------------
// the kernel
// ---------------------------------------------------------------------------------------------------
template <int LS, bool DENSE, class PosT>
__global__ void __launch_bounds__(NT, 1)
jacobian2_kernel(const DevJac m, const DevJacOut o, int mode, int64_t n_states, int64_t tile, int tshift, const double* __restrict__ phi,
                 const double* __restrict__ param, double* __restrict__ out, unsigned long long* __restrict__ sched) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  constexpr int S = 2 * LS, IPW = 32 / LS;
  Smem<LS> sm(smem_raw, m);
  __shared__ int cnt[4];
  __shared__ long long next_tile;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, pr = tid % LS;
  const int ns = m.ns, L = ns - 1, nvar = m.nvar;
  const bool conp = mode == PYJAC_CONP;
  const double conv = conp ? 0.0 : 1.0;
  // ---- once per CTA: what does not depend on the state ------------------------------------------------------------
  for (int i = tid; i < m.nr; i += NT) sm.dn[i] = __ldg(m.dn + i);
  for (int i = tid; i < m.n_groups; i += NT) sm.grp[i] = __ldg(reinterpret_cast<const int4*>(m.groups) + i);
  if (tid < J_NZERO * LS) st2(sm.V + m.ns_max * LS + tid, mk(0.0));
  if (tid < LS) { st2(sm.C + ns * LS + tid, mk(1.0)); st2(sm.G + ns * LS + tid, mk(0.0)); st2(sm.Hh + ns * LS + tid, mk(0.0)); st2(sm.K + ns * LS + tid, mk(0.0)); }
  if (tid < 4) cnt[tid] = 0;
  const int64_t n_tiles = (n_states + S - 1) / S;
  const bool vec = (tile & 1) == 0;
  const int n2 = nvar * nvar;
  const int n_zslices = DENSE ? (n2 + 1023) / 1024 : 0;
  // per-pair scalars of a tile, by the first warp (T, E and the parameter already in registers): double-buffered,
  // the scalars of tile n + 1 are computed while tile n is gathered
  auto write_scalars = [&](D2* sc, D2 T, D2 E_, D2 par) {
    const D2 V = conp ? E_ : par, Pp = conp ? par : E_;
    if (lane < LS) {
      const D2 invT = mk(1.0 / T.a, 1.0 / T.b), lnT = mk(log_lib(T.a), log_lib(T.b)), RT = T * R_GAS;
      const D2 Ctot = mk(Pp.a / RT.a, Pp.b / RT.b);
      st2(sc + SC_T * LS + pr, T); st2(sc + SC_V * LS + pr, V); st2(sc + SC_P * LS + pr, Pp);
      st2(sc + SC_INVT * LS + pr, invT); st2(sc + SC_LNT * LS + pr, lnT); st2(sc + SC_CTOT * LS + pr, Ctot);
      st2(sc + SC_RT * LS + pr, RT); st2(sc + SC_LNP * LS + pr, mk(log_lib(Pp.a), log_lib(Pp.b)));
      st2(sc + SC_LNPRT * LS + pr, mk(log_lib(P_ATM / RT.a), log_lib(P_ATM / RT.b)));
    }
  };
  // this thread's pair of states in tile t (ragged tail: the last state is recomputed, never stored)
  auto pair_of = [&](int64_t t, int64_t& sa, int64_t& sb) { const int64_t s0 = t * S + 2 * pr; sa = min(s0, n_states - 1); sb = min(s0 + 1, n_states - 1); };
  // moles of the species this thread handles in the first trip of the species loop
  const int k_mine = tid / LS;
  auto fetch_moles = [&](int64_t t) {
    int64_t sa, sb; pair_of(t, sa, sb);
    if (k_mine < L) return mk(phi[state_base(sa, tshift, nvar) + (int64_t)(2 + k_mine) * tile], phi[state_base(sb, tshift, nvar) + (int64_t)(2 + k_mine) * tile]);
    return mk(0.0);
  };
  D2* sc_other = sm.sc + J_NSC * LS;
  D2 pn = mk(0.0);
  if ((int64_t)blockIdx.x < n_tiles) {
    pn = fetch_moles(blockIdx.x);
    if (warp == 0) {
      int64_t sa, sb; pair_of(blockIdx.x, sa, sb);
      const double *pha = phi + state_base(sa, tshift, nvar), *phb = phi + state_base(sb, tshift, nvar);
      write_scalars(sm.sc, mk(pha[0], phb[0]), mk(pha[tile], phb[tile]), mk(param[sa], param[sb]));
    }
  }
  __syncthreads();
  for (int64_t tl = blockIdx.x; tl < n_tiles;) {
    if (tid == 0) { next_tile = (long long)gridDim.x + (long long)atomicAdd(sched, 1ull); cnt[2] = 0; cnt[3] = 0; }   // read after the next barrier
    const int64_t s0 = tl * S + 2 * pr;
    const bool va = s0 < n_states, vb = s0 + 1 < n_states;
    const int64_t sa = min(s0, n_states - 1), sb = min(s0 + 1, n_states - 1);
    const double* __restrict__ pha = phi + state_base(sa, tshift, nvar);
    const double* __restrict__ phb = phi + state_base(sb, tshift, nvar);
    Out og;
    og.pa = out + state_base(sa, tshift, o.n_e); og.pb = out + state_base(sb, tshift, o.n_e);
    og.tile = tile; og.va = va; og.vb = vb; og.full = vec && vb;
    // ---- phase 0b: species (C_k = n_k / V, Eq. 6; NASA-7 thermo, R2) ------------------------------------
    {
      const D2 T = ld2(sm.sc + SC_T * LS + pr), V = ld2(sm.sc + SC_V * LS + pr);
      const D2 invT = ld2(sm.sc + SC_INVT * LS + pr), lnT = ld2(sm.sc + SC_LNT * LS + pr);
      const D2 T2 = T * T, T3 = T2 * T, T4 = T3 * T;
      const D2 invV = mk(1.0 / V.a, 1.0 / V.b);
      D2 acc0 = mk(0.0), acc1 = mk(0.0), acc2 = mk(0.0);
      for (int idx = tid; idx < ns * LS; idx += NT) {
        const int k = idx / LS;
        const double* __restrict__ tab = m.nasa + k;               // coefficient-major: tmid, lo[7], hi[7]
        const double tmid = __ldg(tab);
        const bool la = T.a <= tmid, lb = T.b <= tmid;             // low range iff T <= T_mid (R3)
        double ca[7], cb[7];
        if (la == lb) {
#pragma unroll
          for (int c = 0; c < 7; ++c) { ca[c] = __ldg(tab + (size_t)((la ? 1 : 8) + c) * ns); cb[c] = ca[c]; }
        } else {
#pragma unroll
          for (int c = 0; c < 7; ++c) { const double lo = __ldg(tab + (size_t)(1 + c) * ns), hi = __ldg(tab + (size_t)(8 + c) * ns); ca[c] = la ? lo : hi; cb[c] = lb ? lo : hi; }
        }
        auto thermo = [&](const double (&a)[7], double t, double t2, double t3, double t4, double it, double lt, double& cpR, double& dcpR, double& hRT, double& sR) {
          cpR = a[0] + a[1] * t + a[2] * t2 + a[3] * t3 + a[4] * t4;
          dcpR = a[1] + 2.0 * a[2] * t + 3.0 * a[3] * t2 + 4.0 * a[4] * t3;
          hRT = a[0] + a[1] * t * 0.5 + a[2] * t2 * (1.0 / 3.0) + a[3] * t3 * 0.25 + a[4] * t4 * 0.2 + a[5] * it;
          sR = a[0] * lt + a[1] * t + a[2] * t2 * 0.5 + a[3] * t3 * (1.0 / 3.0) + a[4] * t4 * 0.25 + a[6];
        };
        D2 cpR, dcpR, hRT, sR;
        thermo(ca, T.a, T2.a, T3.a, T4.a, invT.a, lnT.a, cpR.a, dcpR.a, hRT.a, sR.a);
        thermo(cb, T.b, T2.b, T3.b, T4.b, invT.b, lnT.b, cpR.b, dcpR.b, hRT.b, sR.b);
        const D2 c = (cpR - conv) * R_GAS;                            // c_p or c_v = c_p - R
        st2(sm.G + idx, hRT - sR);
        st2(sm.Hh + idx, hRT);
        st2(sm.K + idx, c);
        if (k < L) {
          const D2 Ck = (idx == tid ? pn : mk(pha[(int64_t)(2 + k) * tile], phb[(int64_t)(2 + k) * tile])) * invV;
          st2(sm.C + idx, Ck);
          acc0 += Ck; acc1 = fma2(Ck, c, acc1); acc2 = fma2(Ck, dcpR * R_GAS, acc2);
        } else {
          st2(sm.sc + SC_EL * LS + pr, hRT - conv); st2(sm.sc + SC_CL * LS + pr, c); st2(sm.sc + SC_DCL * LS + pr, dcpR * R_GAS);
        }
      }
#pragma unroll
      for (int off = 16; off >= LS; off >>= 1) { acc0 += shfl_xor2(acc0, off); acc1 += shfl_xor2(acc1, off); acc2 += shfl_xor2(acc2, off); }
      if (lane < LS) { st2(sm.red + (warp * J_NRED + 8) * LS + lane, acc0); st2(sm.red + (warp * J_NRED + 9) * LS + lane, acc1); st2(sm.red + (warp * J_NRED + 10) * LS + lane, acc2); }
      // reaction sums of this tile start at zero (per-warp partials, summed by their consumers)
      if (lane < 8 * LS) st2(sm.red + warp * J_NRED * LS + lane, mk(0.0));
    }
    __syncthreads();
    const int64_t tl_next = next_tile;
    if (tid < LS) {
      // the last species: C_Ns from the ideal-gas law
      D2 s0_ = mk(0.0), s1_ = mk(0.0), s2_ = mk(0.0);
      for (int w = 0; w < NW; ++w) { s0_ += ld2(sm.red + (w * J_NRED + 8) * LS + tid); s1_ += ld2(sm.red + (w * J_NRED + 9) * LS + tid); s2_ += ld2(sm.red + (w * J_NRED + 10) * LS + tid); }
      const D2 CL = ld2(sm.sc + SC_CTOT * LS + tid) - s0_;
      st2(sm.C + L * LS + tid, CL);
      st2(sm.sc + SC_D * LS + tid, s1_ + CL * ld2(sm.sc + SC_CL * LS + tid));
      st2(sm.sc + SC_DDDT * LS + tid, s2_ + CL * ld2(sm.sc + SC_DCL * LS + tid));
    }
    __syncthreads();
    for (int b = 0; b <= m.H; ++b) {
      if (b < m.H) {
        // ---- phase 1: reactions of block b ------------------------------------------------------------------------
        // One lane per (reaction, pair, STATE): scalar code, half the registers of a two-state formulation, so that 16
        // warps fit without spills (phase 1 is bound by dependent fp64 latency: it needs the warps, not the sharing of
        // table words between the two states).  16 / LS reactions per chunk; the reactions of the general path come
        // first in the block (they are the expensive ones: longest-processing-time-first).
        const int prs = (lane >> 1) % LS, st = lane & 1;                 // this lane's pair and state
        const double* __restrict__ scd = reinterpret_cast<const double*>(sm.sc);
        auto scv = [&](int i) { return scd[(i * LS + prs) * 2 + st]; };
        const double V = scv(SC_V), invT = scv(SC_INVT), lnT = scv(SC_LNT), Ctot = scv(SC_CTOT), RT = scv(SC_RT), ln_patm_rt = scv(SC_LNPRT);
        const double eL = scv(SC_EL), cL = scv(SC_CL);
        const double ctot_T = Ctot * invT;
        const int r0 = m.blk_r0[b], nrb = m.blk_r0[b + 1] - r0, ng = m.blk_ng[b];
        constexpr int RPC = 16 / LS;                                     // reactions per chunk
        const int n_gchunks = (ng + RPC - 1) / RPC, n_chunks = n_gchunks + (nrb - ng + RPC - 1) / RPC;
        double acc[8];
#pragma unroll
        for (int q = 0; q < 8; ++q) acc[q] = 0.0;
        const double* __restrict__ Cd = reinterpret_cast<const double*>(sm.C) + prs * 2 + st;
        const double* __restrict__ Gd = reinterpret_cast<const double*>(sm.G) + prs * 2 + st;
        const double* __restrict__ Hd = reinterpret_cast<const double*>(sm.Hh) + prs * 2 + st;
        const double* __restrict__ Kd = reinterpret_cast<const double*>(sm.K) + prs * 2 + st;
        double* __restrict__ Vd = reinterpret_cast<double*>(sm.V) + prs * 2 + st;
        for (int chunk = next_chunk(cnt + 0); chunk < n_chunks; chunk = next_chunk(cnt + 0)) {
          const bool general = chunk < n_gchunks;
          const int lr = general ? chunk * RPC + lane / (2 * LS) : ng + (chunk - n_gchunks) * RPC + lane / (2 * LS);
          if (lr >= (general ? ng : nrb)) continue;
          const int r = r0 + lr;
          const uint32_t info = __ldg(m.info + r);
          const uint4 spw = __ldg(reinterpret_cast<const uint4*>(m.sp) + r);
          if (general) {
            double inc[7];
            reaction_general<LS>(m, sm, r, lr, prs, st, conp, info, spw, inc);
#pragma unroll
            for (int q = 0; q < 7; ++q) acc[q] += inc[q];
            continue;
          }
          // fast path: elementary or third-body reaction, all coefficients 1, <= 2 species per side, the last
          // species in no role
          const double rx_lnA = __ldg(m.lnA + r), rx_beta = __ldg(m.beta + r), rx_Ta = __ldg(m.Ta + r), dn = sm.dn[r];
          const int k0 = (spw.x & 0xffffu) * (2 * LS), k1 = (spw.x >> 16) * (2 * LS), k2 = (spw.y >> 16) * (2 * LS), k3 = (spw.z & 0xffffu) * (2 * LS);   // reactants 0, 1; products 3, 4
          const double C0 = Cd[k0], C1 = Cd[k1], C2 = Cd[k2], C3 = Cd[k3];
          const double dh = (Hd[k2] + Hd[k3]) - (Hd[k0] + Hd[k1]);
          const double dc = (Kd[k2] + Kd[k3]) - (Kd[k0] + Kd[k1]);
          const double lnkf = fma(rx_beta, lnT, rx_lnA) - rx_Ta * invT;
          const double lam_f = fma(rx_Ta, invT, rx_beta) * invT;
          const double snu = (double)((int)((info >> JI_SNU_SHIFT) & 31u) - 16);
          const bool rev = info & JI_REV;
          // a4: K_c from the Gibbs polynomials, k_r = k_f / K_c = exp(ln k_f - ln K_c); both exponentials together
          double arg_r = lnkf, lam_r = 0.0;
          if (rev) {
            const double dg = (Gd[k2] + Gd[k3]) - (Gd[k0] + Gd[k1]);
            arg_r = lnkf + dg - snu * ln_patm_rt;
            lam_r = lam_f - (dh - snu) * invT;
          }
          double kf = exp_core(lnkf), kr = exp_core(arg_r);
          if (!(exp_in_range(lnkf) && exp_in_range(arg_r))) { kf = exp_lib(lnkf); kr = exp_lib(arg_r); }
          if (!rev) kr = 0.0;
          const double Rf = kf * (C0 * C1), Rr = kr * (C2 * C3), Rn = Rf - Rr;
          const double dRdT = lam_f * Rf - lam_r * Rr;
          double* __restrict__ Vp = Vd + (spw.w & 0xffffu) * (2 * LS);
          constexpr int SL = 8 * 2 * LS;                                 // doubles between consecutive slots of a reaction
          const int nre = (info >> JI_NREAC_SHIFT) & 3, npr = (info >> JI_NPROD_SHIFT) & 3;
          double c = 1.0, GT = dRdT, MdcdM_R = 0.0, GL = 0.0;
          if ((info & JI_TYPE_MASK) == PYJAC_THIRD_BODY) {
            const int4 ext = __ldg(reinterpret_cast<const int4*>(m.ext) + r);
            const double adef = (info & JI_ADEF) ? 1.0 : 0.0;
            const int si = 2 + nre + (rev ? npr : 0);
            double M = Ctot * adef;
            for (int q0 = 0; q0 < ext.z; q0 += 4) {                       // efficiency list, 4 entries per round trip
              int esp[4]; double ed[4];
#pragma unroll
              for (int q = 0; q < 4; ++q) { esp[q] = q0 + q < ext.z ? __ldg(m.eff_sp + ext.y + q0 + q) : ns; ed[q] = q0 + q < ext.z ? __ldg(m.eff_d + ext.y + q0 + q) : 0.0; }
#pragma unroll
              for (int q = 0; q < 4; ++q) {
                M = fma(ed[q], Cd[esp[q] * (2 * LS)], M);
                if (q0 + q < ext.z) Vp[(si + q0 + q) * SL] = Rn * ed[q];     // dQ/dC_e through [M]: alpha' X, X = R_n
              }
            }
            c = M; GT = M * dRdT; MdcdM_R = M * Rn; GL = Rn * adef;
          }
          const double q = c * Rn;
          const double a_ = c * kf, b_ = c * kr;
          Vp[2 * SL] = a_ * C1;
          if (nre == 2) Vp[3 * SL] = a_ * C0;
          if (rev) {
            Vp[(2 + nre) * SL] = -(b_ * C3);
            if (npr == 2) Vp[(3 + nre) * SL] = -(b_ * C2);
          }
          const double slotT = V * (GT - ctot_T * GL);
          double slotE;
          if (conp) {
            const double of = (double)((info >> JI_OF_SHIFT) & 15), orv = (double)((info >> JI_OR_SHIFT) & 15);
            slotE = q - c * (Rf * of - Rr * orv) - MdcdM_R + Ctot * GL;
          } else {
            slotE = V * (GL / RT);
          }
          Vp[0] = slotT;
          Vp[SL] = slotE;
          const double dEt = RT * (dh - conv * snu - eL * (snu - dn));
          const double dct = dc - cL * (snu - dn);
          reinterpret_cast<double*>(sm.dE)[(lr * LS + prs) * 2 + st] = dEt;
          acc[0] = fma(dEt, q, acc[0]); acc[1] = fma(dn, q, acc[1]); acc[2] = fma(dEt, slotT, acc[2]); acc[3] = fma(dn, slotT, acc[3]);
          acc[4] = fma(dEt, slotE, acc[4]); acc[5] = fma(dn, slotE, acc[5]); acc[6] = fma(dct, q, acc[6]);
        }
        // per-warp partial reaction sums (the barrier below publishes them together with the slots)
        {
          double* __restrict__ redd = reinterpret_cast<double*>(sm.red + warp * J_NRED * LS);
          WarpSum<8, 16, 2 * LS>::run(acc, 0, true, [&](int jv, double x) { if (jv < 7) redd[(jv * LS + prs) * 2 + st] += x; });
        }
        __syncthreads();
        if (tid == 0) cnt[0] = 0;
        if (b == m.H - 1) {
          // every reaction is done.  a10: the four corner entries from the reaction sums (R4-7), by the last warp
          if (warp == NW - 1 && lane < LS) {
            const D2 T = ld2(sm.sc + SC_T * LS + pr), Pp = ld2(sm.sc + SC_P * LS + pr), D = ld2(sm.sc + SC_D * LS + pr);
            const D2 V = ld2(sm.sc + SC_V * LS + pr), Ctot = ld2(sm.sc + SC_CTOT * LS + pr), cL = ld2(sm.sc + SC_CL * LS + pr);
            D2 sums[7];
#pragma unroll
            for (int q = 0; q < 7; ++q) { sums[q] = mk(0.0); for (int w = 0; w < NW; ++w) sums[q] += ld2(sm.red + (w * J_NRED + q) * LS + pr); }
            const D2 dDdT0 = ld2(sm.sc + SC_DDDT * LS + pr);
            const D2 fT = mk(-sums[0].a / D.a, -sums[0].b / D.b);        // f_T = -N / D (Eq. 5)
            D2 JTT, JTE, JET, JEE;
#pragma unroll 1
            for (int h2 = 0; h2 < 2; ++h2) {
              auto pick = [&](D2 x) { return h2 ? x.b : x.a; };
              const double T_ = pick(T), V_ = pick(V), Pp_ = pick(Pp), Ctot_ = pick(Ctot), D_ = pick(D), cL_ = pick(cL), fT_ = pick(fT);
              const double N = pick(sums[0]), Ssum = pick(sums[1]), AT = pick(sums[2]), BT = pick(sums[3]), AE = pick(sums[4]), BE = pick(sums[5]), sumcw = pick(sums[6]);
              const double iV = 1.0 / V_;
              const double dN_dT = AT * iV + sumcw;
              const double dD_dT = pick(dDdT0) - cL_ * Ctot_ / T_;
              const double jTT = -(dN_dT + fT_ * dD_dT) / D_;
              const double dS_dT = BT * iV;
              double dN_dE, dD_dE, dS_dE, jTE, jET, jEE;
              if (conp) {
                const double fE = V_ * (T_ * R_GAS / Pp_ * Ssum + fT_ / T_);
                dN_dE = (AE - N) * iV; dD_dE = -(D_ - Ctot_ * cL_) * iV; dS_dE = (BE - Ssum) * iV;
                jTE = -(dN_dE + fT_ * dD_dE) / D_;
                jET = V_ * (T_ * R_GAS / Pp_ * dS_dT + jTT / T_) + V_ * (R_GAS * Ssum / Pp_ - fT_ / (T_ * T_));
                jEE = V_ * (T_ * R_GAS / Pp_ * dS_dE + jTE / T_) + fE * iV;
              } else {
                dN_dE = AE * iV; dD_dE = cL_ / (R_GAS * T_); dS_dE = BE * iV;
                jTE = -(dN_dE + fT_ * dD_dE) / D_;
                jET = T_ * R_GAS * dS_dT + Pp_ / T_ * jTT + R_GAS * Ssum - Pp_ * fT_ / (T_ * T_);
                jEE = T_ * R_GAS * dS_dE + Pp_ / T_ * jTE + fT_ / T_;
              }
              if (h2) { JTT.b = jTT; JTE.b = jTE; JET.b = jET; JEE.b = jEE; } else { JTT.a = jTT; JTE.a = jTE; JET.a = jET; JEE.a = jEE; }
            }
            og.store((uint32_t)o.d_pos[0], JTT); og.store((uint32_t)o.d_pos[1], JTE); og.store((uint32_t)o.d_pos[2], JET); og.store((uint32_t)o.d_pos[3], JEE);
          }
        }
      }
      // ---- phase 2: pieces of block b (b == H: the final combine wave) -----------------------------------------------
      // The state of the NEXT tile is requested before the last block is gathered: its DRAM latency hides behind the
      // gathers, and the first warp turns T, E and the parameter into the next tile's scalars when it runs out of units.
      D2 nT = mk(1.0), nE = mk(1.0), nPar = mk(1.0);
      const bool fetch_next = b == m.H - 1 && tl_next < n_tiles;
      if (fetch_next) {
        pn = fetch_moles(tl_next);
        if (warp == 0) {
          int64_t na, nb_; pair_of(tl_next, na, nb_);
          const double *qa = phi + state_base(na, tshift, nvar), *qb = phi + state_base(nb_, tshift, nvar);
          nT = mk(qa[0], qb[0]); nE = mk(qa[tile], qb[tile]); nPar = mk(param[na], param[nb_]);
        }
      }
      const int g0 = m.blk_g0[b], n_units = (m.blk_g0[b + 1] - g0) * LS;
      int* counter = cnt + (b < m.H ? 1 : 2);
      if (n_units > 0) {
        int unit = next_chunk(counter);
        while (unit < n_units) {
          const int next = next_chunk(counter);
          const int4 gw = sm.grp[g0 + unit / LS];
          JGroup g;
          g.ent_off = (uint32_t)gw.x; g.piece_off = (uint32_t)gw.y;
          g.nP2 = (uint8_t)(gw.z & 0xff); g.nM2 = (uint8_t)((gw.z >> 8) & 0xff); g.cls = (uint8_t)((gw.z >> 16) & 0xff); g.kind = (uint8_t)((uint32_t)gw.z >> 24);
          g.qsteps = (uint32_t)gw.w;
          gather_unit<LS, PosT>(m, o, sm, g, unit % LS, og, conp, b < m.H ? m.blk_r0[b] : 0);
          unit = next;
        }
      }
      if (fetch_next && warp == 0) write_scalars(sc_other, nT, nE, nPar);
      if (DENSE && b == m.H) {
        // structural zeros, each stored once (no memset pass): slices of 1024 elements, one coalesced mask load each
        for (int z = next_chunk(cnt + 3); z < n_zslices; z = next_chunk(cnt + 3)) {
          const int w0 = z * 32, n_words = (n2 + 31) / 32;
          const uint32_t mine = w0 + lane < n_words ? __ldg(o.nzmask + w0 + lane) : 0xffffffffu;
          for (int q = lane / LS; q < 1024; q += IPW) {
            const uint32_t wj = __shfl_sync(0xffffffffu, mine, q >> 5);
            const int e = z * 1024 + q;
            if (!((wj >> (q & 31)) & 1u) && e < n2) og.store((uint32_t)e, mk(0.0));
          }
        }
      }
      __syncthreads();
      if (tid == 0 && b < m.H) cnt[1] = 0;
    }
    tl = tl_next;
    { D2* t_ = sm.sc; sm.sc = sc_other; sc_other = t_; }
  }
  if (tid == 0 && atomicAdd(sched + 1, 1ull) == (unsigned long long)gridDim.x - 1) { sched[0] = 0; sched[1] = 0; }
}

}  // namespace jac2
}  // namespace pyjac
