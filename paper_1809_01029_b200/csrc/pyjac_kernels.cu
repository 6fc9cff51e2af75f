// fp64 kernels of the hot path for sm_100a (steps a1-a11 of SURVEY.md section 8a / DESIGN.md).
//
// Design: a CTA owns a TILE OF S STATES and keeps every per-state intermediate
// on chip.  All work loops run over (item, state) pairs with the state index fastest inside the warp,
// so every global access of a warp is a run of S consecutive states.
//   phase 0  items = species    : concentrations (Eq. 6-7), NASA-7 thermo, D = sum C_k c_k
//   phase 1  items = reactions  : k_f, K_c, k_r, third-body / falloff c_i, rates of progress and the
//                                 per-reaction partials ("slots") dq_i/dT, dq_i/dE, dQ_i/dC_j -> shared
//                                 memory; reaction-sum reductions for the T and E source terms
//   phase 2  items = nonzeros   : every Jacobian nonzero gathers its static list of slots from shared
//                                 memory, is finished in a register and stored ONCE (no zero-fill +
//                                 "J[idx] += ..." read-modify-write as in PAPER.md L343, no index
//                                 search as in PAPER.md L345)
// No tensor cores: nothing here is a dense contraction.  No fast-math.
#include <cuda_runtime.h>

#include <algorithm>

#include "pyjac_internal.h"
#include "pyjac_math.cuh"

namespace pyjac {

namespace {

// unroll factors / segments per thread of the gathers (measured on C5 / C2 / C3, profiles/r01_sweeps.md)
constexpr int PYJAC_UJ = 4;    // species-row gather, wide groups: segments per thread
constexpr int PYJAC_UC = 2;    // T/E-row gather: segments per thread
constexpr int PYJAC_UNJ = 2;   // entry-loop unroll of the species-row gather (in words = pairs of entries)
constexpr int PYJAC_UNC = 4;   // entry-loop unroll of the T/E-row gather
constexpr int PYJAC_UN1 = 8;   // narrow gather at one state per CTA: segments per thread
constexpr int PYJAC_UQ = 1;    // source-term gather: segments per thread
constexpr int XIT = XPAIR_PAD / 32;   // dense by expansion: warp iterations (of 32 element pairs) per batch
constexpr int ZERO_WARPS = 1;   // warps that stream the zero fill of large dense matrices
constexpr int NT = 512;            // threads per CTA
constexpr int NW = NT / 32;
constexpr int NRED = 10;          // reduction slots: 0-6 reaction sums (phase 1), 7-9 species sums (phase 0)
constexpr int RED0 = 7;
// per-state scalars kept in shared memory
enum { SC_T = 0, SC_V, SC_P, SC_CTOT, SC_SUMC, SC_SUMCC, SC_SUMCDC, SC_D, SC_DDDT, SC_CNS,
       SC_R0, SC_R1, SC_R2, SC_R3, SC_R4, SC_R5, SC_R6, SC_R7, SC_INVT, SC_LNT, SC_LNP, SC_LNPRT, NSC };

__host__ __device__ inline size_t smem_doubles(int ns, int nr, int nslots, int n_part, int n_meta, int S, bool jac) {
  // C[ns+1] (C[ns] = 1: dummy species of unused stoichiometric entries), gh, ec [2(ns+1)] each, ck[ns], slots (+ zero slots)
  size_t per_state = NSC + 6 * (size_t)ns + 5 + (jac ? (size_t)nslots + nr : (size_t)nr) + N_ZERO_SLOTS;
  // n_part: partial sums of split gather lists; n_meta: (offset, width) of every ELL super-group (8 bytes each)
  // Jacobian kernel (persistent CTA): the NASA table [15*ns]
  // and a second c_k array (the second pass of tile n overlaps phase 0 of tile n+1, which rewrites c_k)
  const size_t resident = jac ? 15 * (size_t)ns + (size_t)ns * S : 0;
  return (per_state + n_part) * S + (size_t)NW * NRED * S + n_meta + resident;
}

// Dynamic work distribution inside a CTA: items are sorted by descending cost at create time and warps take the
// next chunk from a shared-memory counter (longest-processing-time-first scheduling); removes the tail in which a
// few warps work on the heaviest reactions / longest gather lists while the others idle.
constexpr int ZERO_WARP_MIN_SLICES = 32;   // dense matrices of >= 32 K elements get a dedicated zero-fill warp
enum { CNT_RX = 0, CNT_J, CNT_J2, CNT_C, CNT_Q, CNT_Z, N_CNT };
__device__ __forceinline__ int next_chunk(int* counter) {
  int c = 0;
  if ((threadIdx.x & 31) == 0) c = atomicAdd(counter, 1);
  return __shfl_sync(0xffffffffu, c, 0);
}

template <int S> __device__ __forceinline__ double red_sum(const double* red, int j, int s);

template <int S> __device__ __forceinline__ double group_sum(double v) {
#pragma unroll
  for (int o = 16; o >= S; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

// Eight per-state sums at once: in the rounds with offset 16, 8, 4 (those >= S) a lane keeps half of its values and
// hands the other half to its partner, so the eight sums cost 4 + 2 + 1 + 1 + 1 = 9 shuffles instead of 40 (S = 1).
// Afterwards a lane holds the sums j0 .. j0 + n - 1 of state lane % S (n = 1 for S <= 4, 2 / 4 / 8 for S = 8 / 16 / 32);
// store(j, value) is called by exactly one lane per (j, state).
template <int S, class StoreF>
__device__ __forceinline__ void group_sum8(double (&v)[8], StoreF store) {
  const int lane = threadIdx.x & 31;
  int j0 = 0;
  constexpr int N16 = S <= 16 ? 4 : 8, N8 = S <= 8 ? N16 / 2 : N16, N4 = S <= 4 ? N8 / 2 : N8;
  if constexpr (S <= 16) {
    const bool up = lane & 16;
#pragma unroll
    for (int i = 0; i < 4; ++i) { const double send = up ? v[i] : v[i + 4], keep = up ? v[i + 4] : v[i]; v[i] = keep + __shfl_xor_sync(0xffffffffu, send, 16); }
    j0 += up ? 4 : 0;
  }
  if constexpr (S <= 8) {
    const bool up = lane & 8;
#pragma unroll
    for (int i = 0; i < 2; ++i) { const double send = up ? v[i] : v[i + 2], keep = up ? v[i + 2] : v[i]; v[i] = keep + __shfl_xor_sync(0xffffffffu, send, 8); }
    j0 += up ? 2 : 0;
  }
  if constexpr (S <= 4) {
    const bool up = lane & 4;
    const double send = up ? v[0] : v[1], keep = up ? v[1] : v[0];
    v[0] = keep + __shfl_xor_sync(0xffffffffu, send, 4);
    j0 += up ? 1 : 0;
  }
  if constexpr (S <= 2) v[0] += __shfl_xor_sync(0xffffffffu, v[0], 2);
  if constexpr (S <= 1) v[0] += __shfl_xor_sync(0xffffffffu, v[0], 1);
  constexpr int PLAIN = (S <= 2 ? 2 : 0) | (S <= 1 ? 1 : 0);     // lane bits summed over without splitting
  if ((lane & PLAIN) == 0) {
#pragma unroll
    for (int i = 0; i < N4; ++i) store(j0 + i, v[i]);
  }
}

// sum over the warps of reduction slot j of state s (partials written by phases01)
template <int S> __device__ __forceinline__ double red_sum(const double* red, int j, int s) {
  double t = 0.0;
#pragma unroll
  for (int w = 0; w < NW; ++w) t += red[(w * NRED + j) * S + s];
  return t;
}

// Outputs are written once and never read back by the kernel: streaming stores (evict-first in L2), so that the
// write stream (up to 1 MB per state in flight per SM) does not push the mechanism tables and gather plans out of L2.
__device__ __forceinline__ void st_out(double* p, double v) { __stcs(p, v); }

__device__ __forceinline__ double apply_sign(double v, uint32_t ent) {
  return __hiloint2double(__double2hiint(v) ^ (int)(ent & SIGN_BIT), __double2loint(v));
}

// block-wide sum of NV per-thread partials per state; result in sc[(first+j)*S + s]
template <int S, int NV>
__device__ __forceinline__ void block_reduce(double (&v)[NV], double* red, double* sc, int first) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
  for (int j = 0; j < NV; ++j) {
    double t = group_sum<S>(v[j]);
    if (lane < S) red[(warp * NRED + j) * S + lane] = t;
  }
  __syncthreads();
  if (threadIdx.x < NV * S) {
    const int j = threadIdx.x / S, s = threadIdx.x % S;
    double t = 0.0;
#pragma unroll
    for (int w = 0; w < NW; ++w) t += red[(w * NRED + j) * S + s];
    sc[(first + j) * S + s] = t;
  }
  __syncthreads();
}

__device__ __forceinline__ double ipow(double x, int n) {   // n in 0..3
  double r = 1.0;
  if (n >= 1) r = x;
  if (n >= 2) r *= x;
  if (n >= 3) r *= x;
  return r;
}
// nu * x^(nu-1), nu in 0..3
__device__ __forceinline__ double dpow(double x, int n) {
  return n == 0 ? 0.0 : (n == 1 ? 1.0 : (n == 2 ? 2.0 * x : 3.0 * x * x));
}

struct Blend { double F, dF_dPr, dF_dT; };

// Troe / SRI blending function and its partial derivatives (R2, R4-5)
__device__ __forceinline__ Blend blend(int type, bool hasT2, const double* __restrict__ fp, double T, double invT, double lnT, double Pr_in) {
  Blend b; b.F = 1.0; b.dF_dPr = 0.0; b.dF_dT = 0.0;
  const double LN10 = 2.302585092994045684, ILN10 = 0.434294481903251828;
  const double Pr = fmax(Pr_in, 1e-300);
  if (type == PYJAC_FALLOFF_TROE) {
    const double a = fp[4], iT3 = 1.0 / fp[5], iT1 = 1.0 / fp[6], T2 = fp[7];
    const double e3 = exp(-T * iT3), e1 = exp(-T * iT1);
    double Fc = (1.0 - a) * e3 + a * e1;
    double dFc = -(1.0 - a) * iT3 * e3 - a * iT1 * e1;
    if (hasT2) { const double e2 = exp(-T2 * invT); Fc += e2; dFc += T2 * invT * invT * e2; }
    const double L = log(Pr) * ILN10, Lc = log(Fc) * ILN10;
    const double n = 0.75 - 1.27 * Lc;
    const double A = L - 0.4 - 0.67 * Lc;
    const double B = n - 0.14 * A;
    const double iB = 1.0 / B;
    const double f = A * iB;
    const double g = 1.0 / (1.0 + f * f);
    b.F = exp(LN10 * Lc * g);
    const double dlogF_df = -2.0 * Lc * f * g * g;
    const double df_dL = n * iB * iB;
    const double df_dLc = (-0.67 * B + 1.1762 * A) * iB * iB;
    b.dF_dPr = b.F * dlogF_df * df_dL / Pr;
    b.dF_dT = b.F * (g + dlogF_df * df_dLc) * dFc / Fc;
  } else if (type == PYJAC_FALLOFF_SRI) {
    const double a = fp[4], bb = fp[5], ic = 1.0 / fp[6], d = fp[7], e = fp[8];
    const double L = log(Pr) * ILN10;
    const double X = 1.0 / (1.0 + L * L);
    const double eb = exp(-bb * invT), ec = exp(-T * ic);
    const double base = a * eb + ec;
    const double dbase = a * bb * invT * invT * eb - ec * ic;
    const double lb = log(base);
    b.F = d * exp(X * lb + e * lnT);
    b.dF_dPr = b.F * lb * (-2.0 * L * X * X) * ILN10 / Pr;
    b.dF_dT = b.F * (X * dbase / base + e * invT);
  }
  return b;
}

// ---------------------------------------------------------------------------------------------------
// phases 0 and 1, shared by the source-term and the Jacobian kernels
// ---------------------------------------------------------------------------------------------------
template <int S, bool JAC>
struct Tile {
  // gh[k*S + s] = (g_k/RT, h_k/RT), ec[k*S + s] = (E~_k, c~_k): two arrays of 16-byte records, so that the 8 lanes of a
  // quarter-warp reading 8 different species can hit 8 different bank groups (one 32-byte record would allow only 4)
  double *sc, *C, *ck, *dE, *P, *red, *part;
  double2 *gh, *ec;
  int2* meta;     // (entry offset, width) of every ELL super-group of the plans this kernel gathers: read per unit
  double *nasa, *phi;   // JAC only (persistent CTA): NASA table, loaded once; phi: the second c_k buffer [ns][S]
  __device__ __forceinline__ Tile(double* smem, int ns, int nr, int nslots, int n_part, int n_meta) {
    sc = smem; gh = reinterpret_cast<double2*>(sc + NSC * S); ec = gh + (ns + 1) * S; C = reinterpret_cast<double*>(ec + (ns + 1) * S); ck = C + (ns + 1) * S; dE = ck + ns * S; P = JAC ? dE + nr * S : dE; red = P + ((JAC ? nslots : nr) + N_ZERO_SLOTS) * S; part = red + NW * NRED * S;
    meta = reinterpret_cast<int2*>(part + n_part * S);
    nasa = reinterpret_cast<double*>(meta + n_meta); phi = nasa + 15 * ns;
    // source kernel: dE unused, P[r] = q_r.  P[nslots ..] (JAC) / P[nr ..]: N_ZERO_SLOTS always-zero slots (ELL padding)
  }
};

// element offset of (element e, state s) in the library layout; base_s precomputed per thread
// tile is a power of two, or tile == ld (then one tile holds every state: s / tile == 0): no 64-bit division
__device__ __forceinline__ int64_t state_base(int64_t s, int64_t tile, int64_t n_e) {
  if (tile & (tile - 1)) return s;
  const int sh = __ffsll((long long)tile) - 1;
  return (((s >> sh) * n_e) << sh) + (s & (tile - 1));
}

// phi_of(e): element e of the state vector of THIS thread's lane (tid % S); par_: that lane's parameter.  The
// analytical kernels read the caller's arrays; the finite-difference kernel adds the perturbation of its column.
// Side job of the dense Jacobian: its DRAM-bound zero fill is done by ONE warp while the other warps work through the
// reaction chunks / gather units (the store queue then blocks that warp only, and the store stream overlaps the
// latency-bound arithmetic).  side(counter, n): true if this warp does the side job instead of taking work items; it
// returns when the items are exhausted (*counter >= n) or the side job is finished.
struct NoSide { __device__ __forceinline__ bool operator()(const int*, int) const { return false; } };

// mid(): called by every thread between the two barriers of phase 0 (the persistent Jacobian kernel finishes the
// previous tile there: its second pass needs a barrier after the gathers, and this one serves).
struct NoMid { __device__ __forceinline__ void operator()() const {} };

// step(): called by every warp before each reaction chunk and each gather unit (the dense-by-expansion kernel streams
// one batch of the PREVIOUS tile's dense matrix out there: different warps are in different kinds of work at any time,
// so the output stream runs alongside the arithmetic instead of in a phase of its own).
struct NoStep { __device__ __forceinline__ void operator()() const {} };

template <int S, bool JAC, class PhiF, class SideF, class MidF, class StepF>
__device__ __forceinline__ void phases01(const DevMech& m, Tile<S, JAC>& t, int mode, PhiF phi_of, double par_,
                                         int* cnt, SideF side, MidF mid, StepF step) {
  const int tid = threadIdx.x;
  const int ns = m.ns, nr = m.nr, L = ns - 1;
  const int s = tid % S;                        // NT % S == 0: a thread keeps its state in every loop
  // ---- phase 0: scalars, species (C_k = n_k / V, Eq. 6; NASA-7 thermo, R2) ------------------------
  // Every thread reads T, E and the parameter itself (same address for the lanes of a state: one broadcast
  // request) so that no barrier separates the state load from the species loop.
  // Nothing that the gathers of the PREVIOUS tile read (work counters, scalars, reaction sums) is written before
  // the first barrier: in the persistent kernel warps enter here while others still gather (idempotent writes excepted).
  if (tid < N_ZERO_SLOTS * S) t.P[(JAC ? m.nslots : nr) * S + tid] = 0.0;   // always-zero slots (ELL padding)
  const double T = phi_of(0), E_ = phi_of(1);
  const double V = mode == PYJAC_CONP ? E_ : par_, Pp = mode == PYJAC_CONP ? par_ : E_;
  const double invT = 1.0 / T, lnT = log(T), RT = R_GAS * T, Ctot = Pp / RT;
  if (tid < S) {
    t.C[ns * S + s] = 1.0;                               // dummy species: unused stoichiometric entries
    t.gh[ns * S + s] = make_double2(0.0, 0.0); t.ec[ns * S + s] = make_double2(0.0, 0.0);
  }
  {
    const double T2 = T * T, T3 = T2 * T, T4 = T3 * T;
    // thermo of the LAST species, evaluated by every thread (cheap, warp-uniform loads): E~_k and c~_k fold the
    // last species in through mass conservation (R1/A1) and need it; saves a second pass and two barriers
    // NASA table (coefficient-major): global memory, or the CTA's shared-memory copy in the persistent Jacobian kernel
    auto nasa = [&](int i) -> double { if constexpr (JAC) return t.nasa[i]; else return __ldg(m.nasa + i); };
    double cL, dcL, eL;
    {
      const int a = L + ((T <= nasa(L)) ? 1 : 8) * ns;
      const double a0 = nasa(a), a1 = nasa(a + ns), a2 = nasa(a + 2 * ns), a3 = nasa(a + 3 * ns), a4 = nasa(a + 4 * ns), a5 = nasa(a + 5 * ns);
      const double cpR = a0 + a1 * T + a2 * T2 + a3 * T3 + a4 * T4;
      const double hRT = a0 + a1 * T * 0.5 + a2 * T2 * (1.0 / 3.0) + a3 * T3 * 0.25 + a4 * T4 * 0.2 + a5 * invT;
      cL = R_GAS * (mode == PYJAC_CONP ? cpR : cpR - 1.0);
      dcL = R_GAS * (a1 + 2.0 * a2 * T + 3.0 * a3 * T2 + 4.0 * a4 * T3);
      eL = hRT - (mode == PYJAC_CONP ? 0.0 : 1.0);
    }
    double acc[3] = {0.0, 0.0, 0.0};
    const double invV = 1.0 / V;
    for (int idx = tid; idx < ns * S; idx += NT) {
      const int k = idx / S;
      // coefficient-major table (entry c of species k at nasa[c * ns + k]): consecutive lanes read consecutive
      // addresses, and BOTH ranges are requested before T is known, so the loads do not wait for the state load
      double a0, a1, a2, a3, a4, a5, a6;
      if constexpr (JAC) {                               // shared-memory table, T already on chip: read one range
        const int b = k + (T <= t.nasa[k] ? 1 : 8) * ns; // low range iff T <= T_mid (R3)
        a0 = t.nasa[b]; a1 = t.nasa[b + ns]; a2 = t.nasa[b + 2 * ns]; a3 = t.nasa[b + 3 * ns]; a4 = t.nasa[b + 4 * ns];
        a5 = t.nasa[b + 5 * ns]; a6 = t.nasa[b + 6 * ns];
      } else {
        const double* __restrict__ a = m.nasa + k;
        double lo[7], hi[7];
        const double tmid = __ldg(a);
#pragma unroll
        for (int c = 0; c < 7; ++c) { lo[c] = __ldg(a + (1 + c) * ns); hi[c] = __ldg(a + (8 + c) * ns); }
        const bool low = T <= tmid;                      // low range iff T <= T_mid (R3); per-lane select
        a0 = low ? lo[0] : hi[0]; a1 = low ? lo[1] : hi[1]; a2 = low ? lo[2] : hi[2]; a3 = low ? lo[3] : hi[3];
        a4 = low ? lo[4] : hi[4]; a5 = low ? lo[5] : hi[5]; a6 = low ? lo[6] : hi[6];
      }
      const double w = __ldg(m.wr + k);
      const double cpR = a0 + a1 * T + a2 * T2 + a3 * T3 + a4 * T4;
      const double dcpR = a1 + 2.0 * a2 * T + 3.0 * a3 * T2 + 4.0 * a4 * T3;
      const double hRT = a0 + a1 * T * 0.5 + a2 * T2 * (1.0 / 3.0) + a3 * T3 * 0.25 + a4 * T4 * 0.2 + a5 * invT;
      const double sR = a0 * lnT + a1 * T + a2 * T2 * 0.5 + a3 * T3 * (1.0 / 3.0) + a4 * T4 * 0.25 + a6;
      const double c = R_GAS * (mode == PYJAC_CONP ? cpR : cpR - 1.0);   // c_p or c_v = c_p - R
      const double e = hRT - (mode == PYJAC_CONP ? 0.0 : 1.0);           // h/RT or u/RT
      t.gh[idx] = make_double2(hRT - sR, hRT);
      // E~_k = E_k - (W_k/W_Ns) E_Ns, c~_k likewise
      t.ec[idx] = k == L ? make_double2(0.0, 0.0) : make_double2(RT * (e - w * eL), c - w * cL);
      t.ck[idx] = c;
      if (k < L) {
        const double Ck = phi_of(2 + k) * invV;
        t.C[idx] = Ck;
        acc[0] += Ck; acc[1] += Ck * c; acc[2] += Ck * (R_GAS * dcpR);
      }
    }
    // block sums; the S finishing threads add the last species: C_Ns from the ideal-gas law
    const int lane = tid & 31, warp = tid >> 5;
#pragma unroll
    for (int j = 0; j < 3; ++j) {
      const double v = group_sum<S>(acc[j]);
      if (lane < S) t.red[(warp * NRED + RED0 + j) * S + lane] = v;
    }
    __syncthreads();
    if (tid >= NT - N_CNT) cnt[NT - 1 - tid] = 0;         // work counters of this tile (last warp: not the finishing threads)
    if (tid < S) {
      t.sc[SC_T * S + s] = T; t.sc[SC_V * S + s] = V; t.sc[SC_P * S + s] = Pp; t.sc[SC_CTOT * S + s] = Ctot;
      t.sc[SC_LNP * S + s] = log(Pp);
      t.sc[SC_LNPRT * S + s] = log(P_ATM / RT);
      double sum[3] = {0.0, 0.0, 0.0};
      for (int w = 0; w < NW; ++w)
#pragma unroll
        for (int j = 0; j < 3; ++j) sum[j] += t.red[(w * NRED + RED0 + j) * S + s];
      const double CL = Ctot - sum[0];
      t.C[L * S + s] = CL;
      t.sc[SC_D * S + s] = sum[1] + CL * cL;
      t.sc[SC_DDDT * S + s] = sum[2] + CL * dcL;
    }
    mid();
    __syncthreads();
  }
  // ---- phase 1: reactions ----------------------------------------------------------------------------
  const double lnP = t.sc[SC_LNP * S + s];
  const double ln_patm_rt = t.sc[SC_LNPRT * S + s];
  const double ctot_T = Ctot * invT;
  double acc[7] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0};
  // One state per CTA: chunks of <= 32 reactions of ONE cost group (table built at create time: HostTables::rxc), in
  // descending cost -- a warp that mixes two reaction types runs both code paths one after the other, and with 16 warps
  // for 70 chunks the longest chunk bounds the phase.  The next chunk's number and span are fetched a chunk ahead.
  // Several states per CTA: chunks of 32 / S reactions are fine-grained enough, plain index arithmetic.
  constexpr bool RXC = S == 1;
  const int n_rx_chunks = RXC ? m.n_rxc[0] : (nr * S + 31) / 32;
  const int2* __restrict__ rxc = reinterpret_cast<const int2*>(m.rxc[0]);
  if (!side(cnt + CNT_RX, n_rx_chunks)) {
  int chunk_next = next_chunk(cnt + CNT_RX);
  int2 span_next = make_int2(0, 0);
  if (RXC && chunk_next < n_rx_chunks) span_next = __ldg(rxc + chunk_next);
  while (chunk_next < n_rx_chunks) {
    step();
    const int chunk = chunk_next;
    const int2 span = span_next;
    chunk_next = next_chunk(cnt + CNT_RX);
    if (RXC && chunk_next < n_rx_chunks) span_next = __ldg(rxc + chunk_next);
    int r;
    if (RXC) {
      r = span.x + (tid & 31);
      if (r >= span.y) continue;
    } else {
      const int i = chunk * 32 + (tid & 31);
      if (i >= nr * S) continue;
      r = i / S;
    }
    const int idx = r * S + s;
    // All per-reaction table words are requested back to back at the top of the iteration and pinned (the empty asm
    // makes every one of them live here), so the reaction costs ONE exposed L2 round trip instead of one per first
    // use further down (the compiler otherwise sinks each load to its consumer: ~3 serialized round trips).
    const int info = __ldg(m.info + r);
    const double rx_lnA = __ldg(m.lnA + r), rx_beta = __ldg(m.beta + r), rx_Ta = __ldg(m.Ta + r), rx_dn = __ldg(m.dn + r);
    const uint4 w0 = __ldg(reinterpret_cast<const uint4*>(m.sp + 8 * r));
    const uint2 w1 = __ldg(reinterpret_cast<const uint2*>(m.sp + 8 * r + 4));
    const int rx_base = JAC ? __ldg(m.slot_base + r) : 0;
    const int e0 = __ldg(m.eff_ptr + r), e1 = __ldg(m.eff_ptr + r + 1);
    const int rx_aux = __ldg(m.aux + r);
    asm volatile("" :: "r"(info), "d"(rx_lnA), "d"(rx_beta), "d"(rx_Ta), "d"(rx_dn), "r"(w0.x), "r"(w0.y), "r"(w0.z), "r"(w0.w),
                 "r"(w1.x), "r"(w1.y), "r"(rx_base), "r"(e0), "r"(e1), "r"(rx_aux));
    const int type = info & INFO_TYPE_MASK;
    const bool rev = info & INFO_REV;
    // ---- fast path (INFO_FAST; the reactions are sorted so that whole chunks take it): elementary or third-body
    // reaction, every coefficient 1, at most two species per side, K_c-based reverse rate, the last species in no role.
    // One code path without the generic ladder: four species records, both exponentials evaluated together by the
    // short-chain exp_core, no powers, no P dependence of k_f.
    if (__all_sync(__activemask(), (info & INFO_FAST) != 0)) {
      const int k0 = w0.x & 0xffff, k1 = w0.y & 0xffff, k3 = w0.w & 0xffff, k4 = w1.x & 0xffff;   // reactants 0, 1; products 3, 4
      const double C0 = t.C[k0 * S + s], C1 = t.C[k1 * S + s], C3 = t.C[k3 * S + s], C4 = t.C[k4 * S + s];
      const double2 g0 = t.gh[k0 * S + s], g1 = t.gh[k1 * S + s], g3 = t.gh[k3 * S + s], g4 = t.gh[k4 * S + s];
      const double2 e0_ = t.ec[k0 * S + s], e1_ = t.ec[k1 * S + s], e3_ = t.ec[k3 * S + s], e4_ = t.ec[k4 * S + s];
      const double dg = (g3.x + g4.x) - (g0.x + g1.x), dh = (g3.y + g4.y) - (g0.y + g1.y);
      const double dEt = (e3_.x + e4_.x) - (e0_.x + e1_.x), dct = (e3_.y + e4_.y) - (e0_.y + e1_.y);
      const double lnkf = fma(rx_beta, lnT, rx_lnA) - rx_Ta * invT;
      const double lam_f = fma(rx_Ta, invT, rx_beta) * invT;
      const double snu = (double)(((info >> INFO_SNU_SHIFT) & 15) - 8);
      double arg_r = lnkf, lam_r = 0.0;
      if (rev) { arg_r = lnkf + dg - snu * ln_patm_rt; lam_r = lam_f - (dh - snu) * invT; }   // a4: k_r = k_f / K_c
      double kf = exp_core(lnkf), kr = exp_core(arg_r);
      if (!(exp_in_range(lnkf) && exp_in_range(arg_r))) { kf = exp(lnkf); kr = exp(arg_r); }
      if (!rev) kr = 0.0;
      const double Rf = kf * (C0 * C1), Rr = kr * (C3 * C4), Rn = Rf - Rr;
      const double dRdT = lam_f * Rf - lam_r * Rr;
      const int nre = (info >> INFO_NREAC_SHIFT) & 3, npr = (info >> INFO_NPROD_SHIFT) & 3;
      double c = 1.0, GT = dRdT, MdcdM_R = 0.0, GL = 0.0;
      if (type == PYJAC_THIRD_BODY) {                      // a5: c = [M]; dQ/dC_e through [M] = alpha' R_n
        const double adef = (info & INFO_ADEF) ? 1.0 : 0.0;
        double M = adef * Ctot;
        const int sl0 = rx_base + 2 + nre + (rev ? npr : 0);
        for (int eb = e0; eb < e1; eb += 4) {
          int esp[4]; double ed[4];
#pragma unroll
          for (int q = 0; q < 4; ++q) { esp[q] = eb + q < e1 ? __ldg(m.eff_sp + eb + q) : ns; ed[q] = eb + q < e1 ? __ldg(m.eff_d + eb + q) : 0.0; }
#pragma unroll
          for (int q = 0; q < 4; ++q) {
            M = fma(ed[q], t.C[esp[q] * S + s], M);
            if (JAC && eb + q < e1) t.P[(sl0 + eb - e0 + q) * S + s] = ed[q] * Rn;
          }
        }
        c = M; GT = M * dRdT; MdcdM_R = M * Rn; GL = adef * Rn;
      }
      const double q = c * Rn;
      acc[0] = fma(dEt, q, acc[0]); acc[1] = fma(rx_dn, q, acc[1]);
      if (!JAC) {
        t.P[idx] = q;
      } else {
        const double a_ = c * kf, b_ = c * kr;
        double* __restrict__ Ps = t.P + rx_base * S + s;
        Ps[2 * S] = a_ * C1;
        if (nre == 2) Ps[3 * S] = a_ * C0;
        if (rev) {
          Ps[(2 + nre) * S] = -(b_ * C4);
          if (npr == 2) Ps[(3 + nre) * S] = -(b_ * C3);
        }
        const double slotT = V * (GT - ctot_T * GL);
        double slotE;
        if (mode == PYJAC_CONP) {
          const double of = (double)((info >> INFO_OF_SHIFT) & 15), orv = (double)((info >> INFO_OR_SHIFT) & 15);
          slotE = q - c * (of * Rf - orv * Rr) - MdcdM_R + Ctot * GL;
        } else {
          slotE = V * (GL / RT);
        }
        Ps[0] = slotT;
        Ps[S] = slotE;
        t.dE[idx] = dEt;
        acc[2] = fma(dEt, slotT, acc[2]); acc[3] = fma(rx_dn, slotT, acc[3]); acc[4] = fma(dEt, slotE, acc[4]);
        acc[5] = fma(rx_dn, slotE, acc[5]); acc[6] = fma(dct, q, acc[6]);
      }
      continue;
    }
    // a3: forward rate constant
    double lnkf, lam_f, dlnk_dP = 0.0;
    if (type <= PYJAC_FALLOFF_SRI) {
      const double beta = rx_beta, Ta = rx_Ta;
      lnkf = rx_lnA + beta * lnT - Ta * invT;
      lam_f = (beta + Ta * invT) * invT;
    } else if (type == PYJAC_PLOG) {
      // table loads are batched (8 independent requests per round trip) instead of one per loop iteration
      const int2 pp = make_int2(__ldg(m.plog_ptr + rx_aux), __ldg(m.plog_ptr + rx_aux + 1));
      const int p0 = pp.x, np = pp.y - pp.x;
      int cnt_le = 0;                                   // number of table pressures <= P
      for (int b = 0; b < np; b += 8) {
        double pq[8];
#pragma unroll
        for (int q = 0; q < 8; ++q) pq[q] = b + q < np ? __ldg(m.plog_P + p0 + b + q) : 1e300;
#pragma unroll
        for (int q = 0; q < 8; ++q) cnt_le += pq[q] <= Pp ? 1 : 0;
      }
      // P <= P_0: first point; P >= P_last: last point; else interval j = last j with P_j <= P (S4)
      const bool interp = cnt_le >= 1 && cnt_le < np && !(cnt_le == 1 && Pp <= __ldg(m.plog_P + p0));
      const int j = cnt_le >= np ? np - 1 : (cnt_le >= 1 ? cnt_le - 1 : 0);
      const int j1 = interp ? j + 1 : j;
      // a pressure level is one entry, or several entries of equal pressure whose rates are summed (R10)
      auto level = [&](int l, double& lnk, double& lam) {
        const int e0 = __ldg(m.plog_ent + p0 + l), e1 = __ldg(m.plog_ent + p0 + l + 1);
        const double bq = __ldg(m.plog_b + e0), Taq = __ldg(m.plog_Ta + e0), lAq = __ldg(m.plog_lnA + e0);
        lnk = lAq + bq * lnT - Taq * invT;
        lam = (bq + Taq * invT) * invT;
        if (e1 - e0 > 1) {
          double ksum = exp(lnk), dsum = ksum * lam;
          for (int e = e0 + 1; e < e1; ++e) {
            const double be = __ldg(m.plog_b + e), Tae = __ldg(m.plog_Ta + e);
            const double ke = exp(__ldg(m.plog_lnA + e) + be * lnT - Tae * invT);
            ksum += ke; dsum += ke * ((be + Tae * invT) * invT);
          }
          lnk = log(ksum); lam = dsum / ksum;
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
      // (T_a(Tr), T_b(Pr) and their derivatives); they are fetched 8 at a time (one round trip per 8, not per 1)
      double cT = 1.0, cTm = 0.0, dT = 0.0, dTm = 0.0;       // T_a(Tr), T_{a-1}, derivatives
      double cP = 1.0, cPm = 0.0, dP = 0.0, dPm = 0.0;
      int ia = 0, ib = 0;
      for (int b = 0; b < n_coef; b += 8) {
        double eq[8];
#pragma unroll
        for (int q = 0; q < 8; ++q) eq[q] = b + q < n_coef ? __ldg(eta + b + q) : 0.0;
#pragma unroll
        for (int q = 0; q < 8; ++q) {
          if (b + q < n_coef) {
            const double e = eq[q];
            lg += e * cT * cP; dlg_dT += e * dT * cP; dlg_dP += e * cT * dP;
            if (++ib == nP) {                    // next row: advance T_a, restart T_b
              ib = 0; ++ia;
              if (ia == 1) { cTm = 1.0; cT = Tr; dTm = 0.0; dT = 1.0; }
              else { const double n1 = 2.0 * Tr * cT - cTm, d1 = 2.0 * cT + 2.0 * Tr * dT - dTm; cTm = cT; cT = n1; dTm = dT; dT = d1; }
              cP = 1.0; cPm = 0.0; dP = 0.0; dPm = 0.0;
            } else if (ib == 1) { cPm = 1.0; cP = Pr_; dPm = 0.0; dP = 1.0; }
            else { const double n1 = 2.0 * Pr_ * cP - cPm, d1 = 2.0 * cP + 2.0 * Pr_ * dP - dPm; cPm = cP; cP = n1; dPm = dP; dP = d1; }
          }
        }
      }
      lnkf = LN10 * lg;
      lam_f = LN10 * dlg_dT * (-2.0 * invT * invT / (iTmax - iTmin));
      dlnk_dP = dlg_dP * 2.0 / (Pp * (lPmax - lPmin));
    }
    const double kf = exp(lnkf);
    // stoichiometry: concentrations, products and one-factor-removed products (no division by C_k: R-S7).
    // Unused entries point at the dummy species ns (C = 1, thermo = 0), so no predicates are needed.
    const uint32_t spw[6] = {w0.x, w0.y, w0.z, w0.w, w1.x, w1.y};
    double pw[6], pm[6];
    double dg = 0.0, dh = 0.0, dEt = 0.0, dct = 0.0;
    // Reactions are sorted so that a warp is (almost always) uniform in "all coefficients are 1": take the vote
    // and branch once, so that the power / multiplicity arithmetic is not executed (if-converted) for the common case.
    // Likewise "no side has a third species" (nearly every reaction): the third positions are skipped warp-wide.
    const bool two = __all_sync(__activemask(), ((info >> INFO_NREAC_SHIFT) & 3) < 3 && ((info >> INFO_NPROD_SHIFT) & 3) < 3);
    if (__all_sync(__activemask(), (info & INFO_SIMPLE) != 0)) {
#pragma unroll
      for (int a = 0; a < 6; ++a) {
        if ((a == 2 || a == 5) && two) { pw[a] = 1.0; pm[a] = 1.0; continue; }
        const int k = spw[a] & 0xffff;
        pw[a] = t.C[k * S + s]; pm[a] = 1.0;
        const double2 gh = t.gh[k * S + s], ec = t.ec[k * S + s];
        if (a < 3) { dg -= gh.x; dh -= gh.y; dEt -= ec.x; dct -= ec.y; }
        else { dg += gh.x; dh += gh.y; dEt += ec.x; dct += ec.y; }
      }
    } else {
#pragma unroll
      for (int a = 0; a < 6; ++a) {
        if ((a == 2 || a == 5) && two) { pw[a] = 1.0; pm[a] = 0.0; continue; }
        const int k = spw[a] & 0xffff, nu = spw[a] >> 16;
        const double Ck = t.C[k * S + s];
        pw[a] = ipow(Ck, nu); pm[a] = dpow(Ck, nu);
        const double2 gh = t.gh[k * S + s], ec = t.ec[k * S + s];
        const double snu = a < 3 ? -(double)nu : (double)nu;
        dg += snu * gh.x; dh += snu * gh.y; dEt += snu * ec.x; dct += snu * ec.y;
      }
    }
    const double Pif = pw[0] * pw[1] * pw[2], Pir = pw[3] * pw[4] * pw[5];
    double kr = 0.0, lam_r = 0.0;
    if (rev) {      // a4: K_c from Gibbs polynomials; k_r = k_f / K_c = exp(ln k_f - ln K_c)
      const double snu = (double)(((info >> INFO_SNU_SHIFT) & 15) - 8);
      if (info & INFO_REVX) {        // explicit reverse Arrhenius parameters (R9): K_c plays no role
        const double lAr = __ldg(m.rev_par + 3 * r), br = __ldg(m.rev_par + 3 * r + 1), Tar = __ldg(m.rev_par + 3 * r + 2);
        kr = exp(lAr + br * lnT - Tar * invT);
        lam_r = (br + Tar * invT) * invT;
      } else {
        kr = exp(lnkf + dg - snu * ln_patm_rt);
        lam_r = lam_f - (dh - snu) * invT;
      }
    }
    const double Rf = kf * Pif, Rr = kr * Pir, Rn = Rf - Rr;
    const double dRdT = lam_f * Rf - lam_r * Rr;
    // a5: third body / falloff
    double c = 1.0, X = 0.0, GT = dRdT, MdcdM_R = 0.0;
    const double adef = (info & INFO_ADEF) ? 1.0 : 0.0;
    if (type >= PYJAC_THIRD_BODY && type <= PYJAC_FALLOFF_SRI) {
      double M = adef * Ctot;                       // sum_k C_k == C_tot by construction of C_Ns
      for (int eb = e0; eb < e1; eb += 4) {           // efficiency list, 4 entries per round trip
        int esp[4]; double ed[4];
#pragma unroll
        for (int q = 0; q < 4; ++q) { esp[q] = eb + q < e1 ? __ldg(m.eff_sp + eb + q) : ns; ed[q] = eb + q < e1 ? __ldg(m.eff_d + eb + q) : 0.0; }
#pragma unroll
        for (int q = 0; q < 4; ++q) M += ed[q] * t.C[esp[q] * S + s];
      }
      if (type == PYJAC_THIRD_BODY) {
        c = M; X = Rn; GT = M * dRdT; MdcdM_R = M * Rn;
      } else {
        // the 10 falloff parameters of the reaction in one batch of 16-byte loads
        double fp[10];
        {
          const double2* __restrict__ f2 = reinterpret_cast<const double2*>(m.fall + 12 * rx_aux);
#pragma unroll
          for (int q = 0; q < 5; ++q) { const double2 v2 = __ldg(f2 + q); fp[2 * q] = v2.x; fp[2 * q + 1] = v2.y; }
          asm volatile("" :: "d"(fp[0]), "d"(fp[1]), "d"(fp[2]), "d"(fp[4]), "d"(fp[5]), "d"(fp[6]), "d"(fp[7]), "d"(fp[8]));
        }
        // falloff: the record holds k_0 and lnkf = ln k_inf.  Chemically activated (R8): the record holds k_inf and
        // lnkf = ln k_0, so the ratio k_0 / k_inf and its temperature derivative change sign in the exponent, and
        // c = F / (1 + Pr) instead of F Pr / (1 + Pr).
        const bool chem = (info & INFO_CHEM) != 0;
        const double b0 = fp[1], Ta0 = fp[2];
        const double lnrat = fp[0] + b0 * lnT - Ta0 * invT - lnkf;
        const double k0_kinf = exp(chem ? -lnrat : lnrat);
        const double Pr = k0_kinf * M;
        const Blend bl = blend(type, info & INFO_T2, fp, T, invT, lnT, Pr);
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
    // reaction-sum reductions (R4-7/8): N = sum dE~_i q_i, S = sum dn~_i q_i
    const double dn = rx_dn;
    acc[0] += dEt * q; acc[1] += dn * q;
    if (!JAC) {
      t.P[idx] = q;
    } else {
      // a8: per-reaction partials -> slots
      const int base = rx_base;
      const int nre = (info >> INFO_NREAC_SHIFT) & 3, npr = (info >> INFO_NPROD_SHIFT) & 3;
      const double a_ = c * kf, b_ = c * kr;
      double GL = adef * X;                          // full dQ_i/dC_Ns
      const double df[3] = {a_ * pm[0] * pw[1] * pw[2], a_ * pw[0] * pm[1] * pw[2], a_ * pw[0] * pw[1] * pm[2]};
      const double dr[3] = {-b_ * pm[3] * pw[4] * pw[5], -b_ * pw[3] * pm[4] * pw[5], -b_ * pw[3] * pw[4] * pm[5]};
      int slot = base + 2;
#pragma unroll
      for (int a = 0; a < 3; ++a)
        if (a < nre) { t.P[(slot++) * S + s] = df[a]; if ((int)(spw[a] & 0xffff) == L) GL += df[a]; }
      if (rev) {
#pragma unroll
        for (int a = 0; a < 3; ++a)
          if (a < npr) { t.P[(slot++) * S + s] = dr[a]; if ((int)(spw[3 + a] & 0xffff) == L) GL += dr[a]; }
      }
      for (int eb = e0; eb < e1; eb += 4) {
        int esp[4]; double ed[4];
#pragma unroll
        for (int q = 0; q < 4; ++q) { esp[q] = eb + q < e1 ? __ldg(m.eff_sp + eb + q) : ns; ed[q] = eb + q < e1 ? __ldg(m.eff_d + eb + q) : 0.0; }
#pragma unroll
        for (int q = 0; q < 4; ++q)
          if (eb + q < e1) {
            const double v = ed[q] * X;
            t.P[(slot++) * S + s] = v;
            if (esp[q] == L) GL += v;
          }
      }
      // chain rule to the state variables (R4-2); E column in Euler-homogeneity form (R4-6)
      const double slotT = V * (GT - ctot_T * GL);
      double slotE;
      if (mode == PYJAC_CONP) {
        const int of = (info >> INFO_OF_SHIFT) & 15, orv = (info >> INFO_OR_SHIFT) & 15;
        slotE = q - c * ((double)of * Rf - (double)orv * Rr) - MdcdM_R + Ctot * GL;
      } else {
        slotE = V * (c * dlnk_dP * Rn + GL / RT);
      }
      t.P[base * S + s] = slotT;
      t.P[(base + 1) * S + s] = slotE;
      t.dE[idx] = dEt;
      acc[2] += dEt * slotT; acc[3] += dn * slotT; acc[4] += dEt * slotE; acc[5] += dn * slotE; acc[6] += dct * q;
    }
  }
  }
  // reaction sums: only the per-warp partials are written here; the single barrier below also publishes the slots.
  // Consumers add the NW partials themselves (red_sum), which saves the second reduction stage and its barrier.
  {
    const int lane = tid & 31, warp = tid >> 5;
    if constexpr (JAC) {
      double v8[8] = {acc[0], acc[1], acc[2], acc[3], acc[4], acc[5], acc[6], 0.0};
      group_sum8<S>(v8, [&](int j, double v) { if (j < 7) t.red[(warp * NRED + j) * S + (lane % S)] = v; });
    } else {
#pragma unroll
      for (int j = 0; j < 2; ++j) {
        const double v = group_sum<S>(acc[j]);
        if (lane < S) t.red[(warp * NRED + j) * S + lane] = v;
      }
    }
  }
  __syncthreads();
}

}  // namespace

namespace {

// ---------------------------------------------------------------------------------------------------
// Gather engine: every output gathers a static list of shared-memory slots.  Items come in order of
// descending list length.  The first n_long items (lists longer than LONG_LIST) are gathered by a whole warp
// (lanes stride the list, shuffle reduction).  The others sit in ELL super-groups of ELL_W = 128 items, lists padded
// to the group's longest and stored entry-major: a thread owns 4 items of a group, so its 4 entry loads per step are
// independent (latency hiding) and the 32 lanes read 32 consecutive entries (coalesced).
//   acc(const int32_t* entry, double (&v)[NACC])      accumulate one entry
//   store(int slot, const double (&v)[NACC])          slot = processing slot (index into the position arrays)
// ---------------------------------------------------------------------------------------------------
// EW = segments per super-group (ELL_W, or ELL_W_NARROW for the narrow tail of the species-row plan); metas points at
// the first of n_groups super-groups, whose first segment has processing slot slot_base.
template <int S, int STRIDE, int NACC, int U, int UNROLL, int EW, class P, class AccF, class PosF, class StoreF, class SideF, class StepF>
__device__ __forceinline__ void gather(const int32_t* __restrict__ ell_ent, const int2* __restrict__ metas, int n_groups,
                                       int slot_base, int* counter, AccF acc, PosF pos_of, StoreF store, SideF side, StepF step) {
  const int lane = threadIdx.x & 31, sub = lane / S;
  constexpr int IPW = 32 / S;                 // segments of one warp per "u"
  // a unit = U * IPW segments of one super-group; a thread owns U segments (U independent loads per step)
  static_assert(EW % (U * IPW) == 0, "super-group must be a whole number of units");
  constexpr int UPG = EW / (U * IPW);         // units per super-group
  const int n_work = n_groups * UPG;
  // metas: (entry offset, padded length) per super-group, in SHARED memory.  Software pipeline: the next unit's
  // number is fetched while the current unit is processed and the output positions are requested before the entry
  // loop, so a unit costs one exposed L2 round trip (its first entries), not three.
  if (side(counter, n_work)) return;
  int unit = next_chunk(counter);
  while (unit < n_work) {
    step();
    const int next = next_chunk(counter);
    const int2 meta = metas[unit / UPG];
    const int sg = unit / UPG;
    const int il0 = (unit % UPG) * (U * IPW) + sub;
    const int slot0 = slot_base + sg * EW + il0;
    P pos[U];
#pragma unroll
    for (int u = 0; u < U; ++u) pos[u] = pos_of(slot0 + u * IPW);
    const int32_t* __restrict__ e = ell_ent + (meta.x + il0) * STRIDE;
    double v[U][NACC];
#pragma unroll
    for (int u = 0; u < U; ++u)
#pragma unroll
      for (int a = 0; a < NACC; ++a) v[u][a] = 0.0;
#pragma unroll UNROLL
    for (int p = 0; p < meta.y; ++p) {
#pragma unroll
      for (int u = 0; u < U; ++u) acc(e + (p * EW + u * IPW) * STRIDE, v[u]);
    }
#pragma unroll
    for (int u = 0; u < U; ++u) store(slot0 + u * IPW, pos[u], v[u]);
    unit = next;
  }
}

// copies the super-group metadata of a plan to shared memory (visible after the next barrier)
__device__ __forceinline__ void load_meta(const DevGather& g, int2* dst) {
  const int2* __restrict__ src = reinterpret_cast<const int2*>(g.sg_meta);
  for (int i = threadIdx.x; i < g.n_sg; i += NT) dst[i] = __ldg(src + i);
}

// second pass over the lists that were split into segments: sum the partial sums, then finish(list, sums)
template <int S, int NACC, class FinishF>
__device__ __forceinline__ void combine(const DevGather& g, const double* __restrict__ part, FinishF finish) {
  const int s = threadIdx.x % S;
  for (int idx = threadIdx.x; idx < g.n_comb * S; idx += NT) {
    const int c = idx / S;
    const int first = g.part_base + NACC * __ldg(g.comb_first + c), n = __ldg(g.comb_nseg + c);
    double v[NACC];
#pragma unroll
    for (int a = 0; a < NACC; ++a) v[a] = 0.0;
    for (int q = 0; q < n; ++q)
#pragma unroll
      for (int a = 0; a < NACC; ++a) v[a] += part[(first + NACC * q + a) * S + s];
    finish(c, v);
  }
}

// ---------------------------------------------------------------------------------------------------
// source terms: Eqs. 3-8
// ---------------------------------------------------------------------------------------------------
template <int S>
__global__ void __launch_bounds__(NT, 1)
source_kernel(const DevMech m, int mode, int64_t n_states, int64_t tile, const double* __restrict__ phi,
              const double* __restrict__ param, double* __restrict__ out) {
  extern __shared__ __align__(16) double smem[];
  Tile<S, false> t(smem, m.ns, m.nr, m.nslots, m.n_part_src, m.qplan.n_sg);
  load_meta(m.qplan, t.meta);
  const int64_t s0 = (int64_t)blockIdx.x * S;
  __shared__ int cnt[N_CNT];
  const int s = threadIdx.x % S;
  const bool valid = s0 + s < n_states;
  const int64_t sg = min(s0 + s, n_states - 1);   // ragged tail: recompute the last valid state, never store
  const int64_t pbase = state_base(sg, tile, m.nvar), obase = pbase;
  phases01<S, false>(m, t, mode, [&](int e) { return phi[pbase + (int64_t)e * tile]; }, param[sg], cnt, NoSide(), NoMid(), NoStep());
  const double V = t.sc[SC_V * S + s];
  // a7: omega_k = sum_i nu_ki q_i (Eq. 4), dn_k/dt = V omega_k (Eq. 3)
  const double* __restrict__ P = t.P;
  gather<S, 1, 1, PYJAC_UQ, 4, ELL_W, int>(m.qplan.ell_ent, t.meta, m.qplan.n_sg, 0, cnt + CNT_Q,
      [&](const int32_t* e, double (&v)[1]) {
        const uint32_t ent = (uint32_t)__ldg(e);
        v[0] += apply_sign(P[(ent & 0x7fffu) * S + s], ent << 16);      // packed: two 16-bit entries per word
        v[0] += apply_sign(P[((ent >> 16) & 0x7fffu) * S + s], ent);
      },
      [&](int slot) { return __ldg(m.q_target + slot); },
      [&](int, int k, const double (&v)[1]) {
        if (k >= 0) { if (valid) st_out(out + obase + (int64_t)(2 + k) * tile, V * v[0]); }
        else if (k <= -2) t.part[(-2 - k) * S + s] = v[0];
      }, NoSide(), NoStep());
  if (m.qplan.n_comb) {
    __syncthreads();
    combine<S, 1>(m.qplan, t.part, [&](int c, const double (&v)[1]) {
      if (valid) st_out(out + obase + (int64_t)(2 + __ldg(m.qc_item + c)) * tile, V * v[0]);
    });
  }
  if (threadIdx.x < S && valid) {
    const double T = t.sc[SC_T * S + s], Pp = t.sc[SC_P * S + s];
    const double fT = -red_sum<S>(t.red, 0, s) / t.sc[SC_D * S + s];          // Eq. 5
    const double Ssum = red_sum<S>(t.red, 1, s);
    const double fE = mode == PYJAC_CONP ? V * (T * R_GAS / Pp * Ssum + fT / T)   // Eq. 8a
                                         : T * R_GAS * Ssum + Pp / T * fT;        // Eq. 8b
    st_out(out + obase, fT);
    st_out(out + obase + tile, fE);
  }
}

// ---------------------------------------------------------------------------------------------------
// First-order forward finite-difference Jacobian -- the paper's own comparison baseline (Fig. 12),
// DESIGN.md R7:   J(i, c) ~ (f_i(phi + h_c e_c) - f_i(phi)) / h_c,   h_c = fl(phi_c + fma(rel, |phi_c|, abs)) - phi_c.
// One CTA per state.  The S lanes of the tile are S perturbed copies of that state: lane s of pass p evaluates the
// source terms at column c = p*S + s - 1; c = -1 (lane 0 of pass 0) is the unperturbed state.  n_var + 1 source
// evaluations per state, against one analytical evaluation: that ratio is what Fig. 12 shows.
// ---------------------------------------------------------------------------------------------------
template <int S>
__global__ void __launch_bounds__(NT, 1)
fd_kernel(const DevMech m, int mode, int ofmt, double rel, double ab, int64_t tile, int64_t n_e,
          const double* __restrict__ phi, const double* __restrict__ param, double* __restrict__ out) {
  extern __shared__ __align__(16) double smem[];
  Tile<S, false> t(smem, m.ns, m.nr, m.nslots, m.n_part_src, m.qplan.n_sg);
  load_meta(m.qplan, t.meta);
  double* __restrict__ f0 = reinterpret_cast<double*>(t.meta + m.qplan.n_sg);   // f(phi)           [nvar]
  double* __restrict__ fc = f0 + m.nvar;                      // f(phi + h_c e_c) [nvar][S]
  __shared__ int cnt[N_CNT];
  const int tid = threadIdx.x, s = tid % S, nvar = m.nvar;
  const int64_t sg = blockIdx.x;
  const int64_t pbase = state_base(sg, tile, nvar), obase = state_base(sg, tile, n_e);
  const double par = param[sg];
  const int n_pass = (nvar + 1 + S - 1) / S;
  for (int pass = 0; pass < n_pass; ++pass) {
    const int c_raw = pass * S + s - 1;
    const int c = c_raw < nvar ? c_raw : -1;                  // lanes past the last column repeat the base state
    double x = 0.0, xp = 0.0;
    if (c >= 0) { x = phi[pbase + (int64_t)c * tile]; xp = x + fma(rel, fabs(x), ab); }
    phases01<S, false>(m, t, mode, [&](int e) { const double v = phi[pbase + (int64_t)e * tile]; return e == c ? xp : v; },
                       par, cnt, NoSide(), NoMid(), NoStep());
    const double V = t.sc[SC_V * S + s];
    const double* __restrict__ P = t.P;
    gather<S, 1, 1, PYJAC_UQ, 4, ELL_W, int>(m.qplan.ell_ent, t.meta, m.qplan.n_sg, 0, cnt + CNT_Q,
        [&](const int32_t* e, double (&v)[1]) {
          const uint32_t ent = (uint32_t)__ldg(e);
          v[0] += apply_sign(P[(ent & 0x7fffu) * S + s], ent << 16);      // packed: two 16-bit entries per word
          v[0] += apply_sign(P[((ent >> 16) & 0x7fffu) * S + s], ent);
        },
        [&](int slot) { return __ldg(m.q_target + slot); },
        [&](int, int k, const double (&v)[1]) {
          if (k >= 0) fc[(2 + k) * S + s] = V * v[0];
          else if (k <= -2) t.part[(-2 - k) * S + s] = v[0];
        }, NoSide(), NoStep());
    if (m.qplan.n_comb) {
      __syncthreads();
      combine<S, 1>(m.qplan, t.part, [&](int q, const double (&v)[1]) { fc[(2 + __ldg(m.qc_item + q)) * S + s] = V * v[0]; });
    }
    if (tid < S) {
      const double T = t.sc[SC_T * S + s], Pp = t.sc[SC_P * S + s];
      const double fT = -red_sum<S>(t.red, 0, s) / t.sc[SC_D * S + s];          // Eq. 5
      const double Ssum = red_sum<S>(t.red, 1, s);
      fc[s] = fT;
      fc[S + s] = mode == PYJAC_CONP ? V * (T * R_GAS / Pp * Ssum + fT / T)      // Eq. 8a
                                     : T * R_GAS * Ssum + Pp / T * fT;           // Eq. 8b
    }
    __syncthreads();
    if (pass == 0) {
      for (int i = tid; i < nvar; i += NT) f0[i] = fc[i * S];
      __syncthreads();
    }
    if (c >= 0) {
      const double h = xp - x;                                // the step actually taken
      if (ofmt >= OUT_DENSE_C) {
        for (int i = tid / S; i < nvar; i += NT / S) {
          const int64_t e = ofmt == OUT_DENSE_C ? (int64_t)i * nvar + c : (int64_t)c * nvar + i;
          st_out(out + obase + e * tile, (fc[i * S + s] - f0[i]) / h);
        }
      } else {                                                // the handle's pattern, walked by columns
        const int p1 = __ldg(m.csc_ptr + c + 1);
        for (int p = __ldg(m.csc_ptr + c) + tid / S; p < p1; p += NT / S) {
          const int i = __ldg(m.csc_idx + p);
          const int64_t e = ofmt == OUT_CSC ? p : __ldg(m.csc2csr + p);
          st_out(out + obase + e * tile, (fc[i * S + s] - f0[i]) / h);
        }
      }
    }
    __syncthreads();                                          // fc, the slots and the work counters are reused
  }
}

// ---------------------------------------------------------------------------------------------------
// Jacobian (sparse CSR / CSC value order or dense 'C' / 'F'), Eq. 9
// ---------------------------------------------------------------------------------------------------
// MODE 0: sparse values.  MODE 1: dense, nonzeros stored at their dense positions + bitmap-driven zero fill.
// MODE 2 (one state per CTA, state-major layout, large matrices): dense by EXPANSION -- the gathers write the sparse
// values (CSR order for 'C', CSC order for 'F': the order of the set bits of the dense bitmap) into the CTA's scratch
// buffer of the tile's parity (L2-resident), and the dense matrix is streamed out while the NEXT tile is computed:
// element e = bit set ? scratch[rank(e)] : 0, in 16-byte pairs with coalesced streaming stores (expand_batch below).
// Every 32-byte sector of the output is written exactly once and completely (MODE 1 writes the zeros and the nonzeros
// of a sector at different times and pays a DRAM read-modify-write for most of them: 1.46 x the algorithmic traffic).
template <int S, int MODE>
__global__ void __launch_bounds__(NT, 1)
jacobian_kernel(const DevMech m, const DevPlan pl, int mode, int64_t n_states, int64_t tile, const double* __restrict__ phi,
                const double* __restrict__ param, double* __restrict__ out, unsigned long long* __restrict__ sched) {
  constexpr bool DENSE = MODE == 1, EXPAND = MODE == 2;
  static_assert(!EXPAND || S == 1, "dense by expansion: one state per CTA");
  // values of the gathers: streaming stores to the caller's array, but write-back stores to the expansion scratch
  // (it is read again a tile later and must stay in L2)
  auto st_g = [](double* q, double v) { if constexpr (MODE == 2) *q = v; else st_out(q, v); };
  extern __shared__ __align__(16) double smem[];
  Tile<S, true> t(smem, m.ns, m.nr, m.nslots, m.n_part_jac, m.cplan.n_sg + pl.jplan.n_sg);
  // PERSISTENT CTA: the grid is one CTA per SM (x occupancy); a CTA starts with tile blockIdx.x and takes further
  // tiles from a global counter (sched[0]; dynamic, because the SMs of the two dies do not run at the same speed when
  // the output stream loads the memory system).  sched[1] counts finished CTAs: the last one resets both words.
  // What does not depend on the state is brought on chip once (gather metadata, NASA table).  Each thread loads the
  // state-vector elements it needs in phase 0 of the NEXT tile into registers right after phase 1, so their DRAM
  // latency hides behind the gathers.  Three barriers per tile: two in phase 0, one after phase 1.  There is none after
  // the gathers: a warp that runs out of gather units starts phase 0 of the next tile, and the second pass over the
  // split lists of tile n runs between the two phase-0 barriers of tile n+1 (the first of them tells it that every
  // partial sum is there).  Phase 0 therefore writes nothing the gathers read before its first barrier; c_k, which the
  // T-row entries of the second pass need, is double-buffered.
  load_meta(m.cplan, t.meta);
  load_meta(pl.jplan, t.meta + m.cplan.n_sg);
  __shared__ int cnt[N_CNT];
  const int tid = threadIdx.x, s = tid % S;
  const int L = m.ns - 1;
  for (int i = tid; i < 15 * m.ns; i += NT) t.nasa[i] = __ldg(m.nasa + i);
  const int64_t n_tiles = (n_states + S - 1) / S;
  // this thread's inputs of phase 0: T, E, the parameter and the moles of species tid / S (first trip of the species loop)
  const int e_mine = tid / S < L ? 2 + tid / S : 0;
  double pT, pE, pPar, pN;
  auto fetch_state = [&](int64_t tl) {
    const int64_t sp = min(tl * S + s, n_states - 1);
    const double* __restrict__ src = phi + state_base(sp, tile, m.nvar);
    pT = src[0]; pE = src[tile]; pN = src[(int64_t)e_mine * tile]; pPar = param[sp];
  };
  fetch_state(blockIdx.x);
  __syncthreads();                                 // NASA table and gather metadata are in place
  double* const ck_buf[2] = {t.ck, reinterpret_cast<double*>(t.phi)};
  __shared__ long long next_tile;
  int parity = 0;
  // context of the previous tile for its deferred second pass
  double* prev_gout = out;
  bool prev_valid = false; int64_t prev_obase = 0; double prev_fT = 0.0, prev_iDV = 0.0, prev_cS = 0.0, prev_cT = 0.0, prev_cL = 0.0;
  const double* prev_ck = t.ck;
  const int nJ2 = pl.jplan.n_comb * S, nC2 = m.cplan.n_comb * S;
  // second pass over the split lists of both plans in ONE index space, with every table word (first partial, count,
  // output positions) requested before the partial sums are added
  auto second_pass = [&]() {
    const double* __restrict__ part = t.part;
    for (int idx = tid; idx < nJ2 + nC2; idx += NT) {
      if (idx < nJ2) {
        const int c = idx / S;
        const int first = pl.jplan.part_base + __ldg(pl.jplan.comb_first + c), n = __ldg(pl.jplan.comb_nseg + c);
        const int pos = __ldg(pl.jc_pos + c);
        double v = 0.0;
        for (int q = 0; q < n; ++q) v += part[(first + q) * S + s];
        if (prev_valid) st_g(prev_gout + prev_obase + (int64_t)pos * tile, v);
      } else {
        const int c = (idx - nJ2) / S;
        const int first = m.cplan.part_base + 2 * __ldg(m.cplan.comb_first + c), n = __ldg(m.cplan.comb_nseg + c);
        const int j = __ldg(m.cc_item + c);
        const int2 pos = __ldg(reinterpret_cast<const int2*>(pl.cc_pos) + c);
        double v0 = 0.0, v1 = 0.0;
        for (int q = 0; q < n; ++q) { v0 += part[(first + 2 * q) * S + s]; v1 += part[(first + 2 * q + 1) * S + s]; }
        if (prev_valid) {
          const double JT = -(v0 + prev_fT * (prev_ck[j * S + s] - prev_cL)) * prev_iDV;
          st_g(prev_gout + prev_obase + (int64_t)pos.x * tile, JT);
          st_g(prev_gout + prev_obase + (int64_t)pos.y * tile, prev_cS * v1 + prev_cT * JT);
        }
      }
    }
  };
  const int nn2 = m.nvar * m.nvar;
  // dense by expansion: the PREVIOUS tile's dense matrix from its sparse values in the scratch buffer, in batches of XIT
  // warp iterations taken from the work counter CNT_Z by every warp: one before each reaction chunk / gather unit of
  // the current tile (step), the rest after the tile's gathers.  The matrix's elements are taken in PAIRS that are
  // 16-byte aligned in the output (pair p = elements 2p - sh, 2p - sh + 1; sh = 1 if the matrix starts on an odd
  // double); a warp iteration covers 32 consecutive pairs (512 contiguous bytes): a lane loads its pair's table word
  // (coalesced; rank << 2 | present bits), the values of the present elements from the scratch (L2) and writes one
  // 16-byte streaming store.  No staging, no intra-warp synchronisation; every 32-byte sector is written once.
  const int n_xb = EXPAND ? ((nn2 + 2) / 2 + XPAIR_PAD - 1) / XPAIR_PAD : 0;
  const double* x_scr = nullptr; double* x_dst = nullptr;
  bool x_more = false;
  auto expand_batch = [&](int b) {
    const int sh = (int)((reinterpret_cast<uintptr_t>(x_dst) >> 3) & 1);
    const int p0 = b * XPAIR_PAD + (tid & 31);
    const int32_t* __restrict__ xp = pl.xpair[sh] + p0;
    int32_t c[XIT];
#pragma unroll
    for (int q = 0; q < XIT; ++q) c[q] = __ldg(xp + q * 32);        // (the table is padded: no bound)
    double va[XIT], vb[XIT];
#pragma unroll
    for (int q = 0; q < XIT; ++q) {
      const double* __restrict__ v = x_scr + (c[q] >> 2);
      va[q] = 0.0; vb[q] = 0.0;
      if (c[q] & 1) va[q] = __ldcg(v);
      if (c[q] & 2) vb[q] = __ldcg(v + (c[q] & 1));
    }
    double* __restrict__ d = x_dst + 2 * p0 - sh;
#pragma unroll
    for (int q = 0; q < XIT; ++q) {
      const int e1 = 2 * (p0 + q * 32) - sh;
      if (e1 >= 0 && e1 + 1 < nn2) __stcs(reinterpret_cast<double2*>(d + q * 64), make_double2(va[q], vb[q]));
      else if (e1 < 0) st_out(x_dst, vb[q]);                      // the odd head element
      else if (e1 < nn2) st_out(x_dst + e1, va[q]);               // the odd tail element
    }
  };
  auto step = [&]() {
    if constexpr (EXPAND) {
      if (x_more) {
        const int b = next_chunk(cnt + CNT_Z);
        if (b < n_xb) expand_batch(b); else x_more = false;
      }
    }
  };
  bool have_prev = false;
  for (int64_t tl = blockIdx.x, tl_next; tl < n_tiles; tl = tl_next, parity ^= 1) {
  unsigned long long ticket = 0;
  if (tid == 0) ticket = atomicAdd(sched, 1ull);   // its latency hides behind the species loop; published in mid()
  t.ck = ck_buf[parity];
  // (with several states per CTA the sparse kernel derives these again after phase 1 instead of keeping them in
  // registers across it: C2 -2.7 %, C3 -3.6 %; at one state per CTA the same change cost 0.4 %)
  const int64_t s0_a = tl * S;
  const bool valid_a = S == 1 || s0_a + s < n_states;   // one state per tile: every tile is a valid state
  const int64_t sg = min(s0_a + s, n_states - 1);   // ragged tail: recompute the last valid state, never store
  constexpr bool REDERIVE = !DENSE && S > 1;
  const int64_t obase_a = REDERIVE || EXPAND ? 0 : state_base(sg, tile, pl.n_e);
  // where the gathers store: the caller's array, or (dense by expansion) this CTA's scratch buffer of the tile's parity
  double* const gout = EXPAND ? pl.scratch + ((size_t)blockIdx.x * 2 + parity) * (size_t)pl.n_e : out;
  bool valid = valid_a; int64_t obase = obase_a;
  // dense output: structural zeros, each stored once (no memset pass), in slices of 32 bitmap words (1024 elements:
  // one coalesced mask load, then 32 coalesced predicated store instructions at S = 1).  For large matrices the
  // last warp streams the slices while the others compute (see NoSide above); what is left is shared at the end.
  const int n2 = m.nvar * m.nvar;
  const int n_zslices = DENSE ? (n2 + 1023) / 1024 : 0;
  auto zero_slice = [&](int slice) {
    if (S == 1) {
      const int lane = tid & 31, w0 = slice * 32, n_words = (n2 + 31) / 32;
      const uint32_t mine = w0 + lane < n_words ? __ldg(pl.nzmask + w0 + lane) : 0xffffffffu;
#pragma unroll 8
      for (int j = 0; j < 32; ++j) {
        const uint32_t wj = __shfl_sync(0xffffffffu, mine, j);
        const int e = (w0 + j) * 32 + lane;
        if (!((wj >> lane) & 1u) && e < n2 && valid) st_out(out + obase + (int64_t)e * tile, 0.0);
      }
    } else {
      for (int q = (tid & 31) / S; q < 1024; q += 32 / S) {
        const int e = slice * 1024 + q;
        if (e < n2 && !((__ldg(pl.nzmask + (e >> 5)) >> (e & 31)) & 1u) && valid) st_out(out + obase + (int64_t)e * tile, 0.0);
      }
    }
  };
  const bool zero_warp = DENSE && n_zslices >= ZERO_WARP_MIN_SLICES && (tid >> 5) >= NW - ZERO_WARPS;
  auto side = [&](const int* counter, int n) -> bool {
    if constexpr (EXPAND) {
      return false;
    } else if constexpr (!DENSE) {
      return false;
    } else {
      if (!zero_warp) return false;
      while (*reinterpret_cast<const volatile int*>(counter) < n) {
        const int z = next_chunk(cnt + CNT_Z);
        if (z >= n_zslices) break;
        zero_slice(z);
      }
      return true;
    }
  };
  {
    const double cT_ = pT, cE_ = pE, cN_ = pN, cPar_ = pPar;
    phases01<S, true>(m, t, mode,
        [&](int e) {
          if (e == 0) return cT_;
          if (e == 1) return cE_;
          if (e == e_mine) return cN_;
          return phi[state_base(sg, tile, m.nvar) + (int64_t)e * tile];     // species loops of more than one trip
        },
        cPar_, cnt, side,
        [&]() {
          if (tid == 0) next_tile = (long long)gridDim.x + (long long)ticket;
          if (have_prev && nJ2 + nC2 > 0) second_pass();
        }, step);
  }
  tl_next = next_tile;
  if (tl_next < n_tiles) fetch_state(tl_next);
  if constexpr (REDERIVE) {
    int64_t tl_b = tl;
    asm volatile("" : "+l"(tl_b));                 // opaque: not a value to keep alive across phase 1
    const int64_t sb = tl_b * S + s;
    valid = sb < n_states;
    obase = state_base(min(sb, n_states - 1), tile, pl.n_e);
  }
  const double T = t.sc[SC_T * S + s], V = t.sc[SC_V * S + s], Pp = t.sc[SC_P * S + s], D = t.sc[SC_D * S + s];
  const double N = red_sum<S>(t.red, 0, s);
  const double fT = -N / D;
  const double cL = t.ck[L * S + s];
  // a10: the four corner entries from the phase-1 reductions (R4-7), by the last warp (it has no item of
  // the second pass).  With several states per CTA they are done BEFORE the gathers (that warp joins the dynamically
  // scheduled gather a little late instead of leaving a serial tail); at one state per CTA the tail measured shorter.
  auto corners = [&]() {
    if ((tid >> 5) == NW - 1 && (tid & 31) < S && valid) {      // the last warp: it has no item of the second pass
      const double Ctot = t.sc[SC_CTOT * S + s];
      const double Ssum = red_sum<S>(t.red, 1, s);
      const double AT = red_sum<S>(t.red, 2, s), BT = red_sum<S>(t.red, 3, s), AE = red_sum<S>(t.red, 4, s), BE = red_sum<S>(t.red, 5, s);
      const double sumcw = red_sum<S>(t.red, 6, s);
      const double iV = 1.0 / V;
      const double dN_dT = AT * iV + sumcw;
      const double dD_dT = t.sc[SC_DDDT * S + s] - cL * Ctot / T;
      const double JTT = -(dN_dT + fT * dD_dT) / D;
      const double dS_dT = BT * iV;
      double dN_dE, dD_dE, dS_dE, JET, JEE, JTE;
      if (mode == PYJAC_CONP) {
        const double fE = V * (T * R_GAS / Pp * Ssum + fT / T);
        dN_dE = (AE - N) * iV; dD_dE = -(D - Ctot * cL) * iV; dS_dE = (BE - Ssum) * iV;
        JTE = -(dN_dE + fT * dD_dE) / D;
        JET = V * (T * R_GAS / Pp * dS_dT + JTT / T) + V * (R_GAS * Ssum / Pp - fT / (T * T));
        JEE = V * (T * R_GAS / Pp * dS_dE + JTE / T) + fE * iV;
      } else {
        dN_dE = AE * iV; dD_dE = cL / (R_GAS * T); dS_dE = BE * iV;
        JTE = -(dN_dE + fT * dD_dE) / D;
        JET = T * R_GAS * dS_dT + Pp / T * JTT + R_GAS * Ssum - Pp * fT / (T * T);
        JEE = T * R_GAS * dS_dE + Pp / T * JTE + fT / T;
      }
      gout[obase + (int64_t)pl.d_pos[0] * tile] = JTT;
      gout[obase + (int64_t)pl.d_pos[1] * tile] = JTE;
      gout[obase + (int64_t)pl.d_pos[2] * tile] = JET;
      gout[obase + (int64_t)pl.d_pos[3] * tile] = JEE;
    }
  };
  corners();     // before the gathers: that warp joins the dynamically scheduled gather a little late, no serial tail
  const double* __restrict__ P = t.P;
  // The T/E-row gather goes FIRST: it has few, long units; warps that finish it early move on to the many short
  // units of the species rows (no barrier in between), so its latency tail is hidden behind them.
  // a10: T and E rows, species columns: gather over reactions with the per-state weights dE~_i, dn~_i
  //   J[T][j] = -(sum_i dE~_i g_ij + f_T (c_j - c_Ns)) / (D V);  J[E][j] = cS sum_i dn~_i g_ij + cT J[T][j]
  const double iDV = 1.0 / (D * V);
  const double cS = mode == PYJAC_CONP ? T * R_GAS / Pp : T * R_GAS / V;
  const double cT = mode == PYJAC_CONP ? V / T : Pp / T;
  const double* __restrict__ dE = t.dE;
  gather<S, 4, 2, PYJAC_UC, PYJAC_UNC, ELL_W, int4>(m.cplan.ell_ent, t.meta, m.cplan.n_sg, 0, cnt + CNT_C,
      [&](const int32_t* e, double (&v)[2]) {
        const int4 pr = __ldg(reinterpret_cast<const int4*>(e));      // slot | sign, reaction, dn~ (2 words)
        const uint32_t ent = (uint32_t)pr.x;
        const double x = apply_sign(P[(ent & ~SIGN_BIT) * S + s], ent);
        v[0] += dE[pr.y * S + s] * x;
        v[1] += __hiloint2double(pr.w, pr.z) * x;
      },
      [&](int slot) {                                     // (T, j) position or partial code, (E, j) position, column j:
        const int2 pp = __ldg(reinterpret_cast<const int2*>(pl.c_pos) + slot);   // all requested before the entry loop
        return make_int4(pp.x, pp.y, __ldg(m.c_item + slot), 0);
      },
      [&](int, int4 pp, const double (&v)[2]) {
        if (pp.x >= 0) {
          if (valid) {
            const double JT = -(v[0] + fT * (t.ck[pp.z * S + s] - cL)) * iDV;
            st_g(gout + obase + (int64_t)pp.x * tile, JT);
            st_g(gout + obase + (int64_t)pp.y * tile, cS * v[1] + cT * JT);
          }
        } else if (pp.x <= -2) {
          const int pi = m.cplan.part_base + 2 * (-2 - pp.x);
          t.part[pi * S + s] = v[0]; t.part[(pi + 1) * S + s] = v[1];
        }
      }, side, step);
  // a9: species rows.  Block entries J[k][j] = sum_i nu_ki (Ghat^j_i - Ghat^Ns_i); T and E columns
  // J[k][T] = sum_i nu_ki slotT_i, J[k][E] = sum_i nu_ki slotE_i.  Every nonzero is finished in a register and
  // stored once.
  {
    auto accJ = [&](const int32_t* e, double (&v)[1]) {
      const uint32_t ent = (uint32_t)__ldg(e);
      v[0] += apply_sign(P[(ent & 0x7fffu) * S + s], ent << 16);      // packed: two 16-bit entries per word
      v[0] += apply_sign(P[((ent >> 16) & 0x7fffu) * S + s], ent);
    };
    double* __restrict__ out_s = gout + obase;
    auto posJ = [&](int slot) { const int p = __ldg(pl.j_pos + slot); return valid || p < 0 ? p : -1; };   // ragged tail: store nothing
    auto storeJ = [&](int, int pos, const double (&v)[1]) {
      if (pos >= 0) st_g(out_s + (int64_t)pos * tile, v[0]);
      else if (pos <= -2) t.part[(-2 - pos) * S + s] = v[0];
    };
    auto storeN = [&](int, int pos, const double (&v)[1]) {      // narrow tail: whole lists only (see build_gather)
      if (pos >= 0) st_g(out_s + (int64_t)pos * tile, v[0]);
    };
    const int2* metaJ = t.meta + m.cplan.n_sg;
    const int n_wide = pl.jplan.n_wide;
    gather<S, 1, 1, PYJAC_UJ, PYJAC_UNJ, ELL_W, int>(pl.jplan.ell_ent, metaJ, n_wide, 0, cnt + CNT_J, accJ, posJ, storeJ, side, step);
    // the narrow tail (lists of one or two entries: most nonzeros of a sparse mechanism): 16 segments per thread
    gather<S, 1, 1, (S == 1 && !DENSE ? PYJAC_UN1 : ELL_W_NARROW / 32), 1, ELL_W_NARROW, int>(pl.jplan.ell_ent, metaJ + n_wide, pl.jplan.n_sg - n_wide, n_wide * ELL_W,
                                              cnt + CNT_J2, accJ, posJ, storeN, side, step);
  }
  if (DENSE)                                      // whatever is left of the zero fill
    for (int z = next_chunk(cnt + CNT_Z); z < n_zslices; z = next_chunk(cnt + CNT_Z)) zero_slice(z);
  prev_gout = gout;
  have_prev = true; prev_valid = valid; prev_obase = obase; prev_fT = fT; prev_iDV = iDV; prev_cS = cS; prev_cT = cT; prev_cL = cL;
  prev_ck = t.ck;
  if constexpr (EXPAND) {
    while (x_more) step();                       // what is left of the previous tile's dense matrix
    x_scr = gout; x_dst = out + tl * (int64_t)nn2;
    x_more = true;                               // (the counter is reset in the next tile's phase 0, behind a barrier)
  }
  }  // tiles of this CTA
  if (have_prev && nJ2 + nC2 > 0) {            // the last tile's second pass
    __syncthreads();
    second_pass();
  }
  if constexpr (EXPAND) {
    if (have_prev) {                             // the last tile's dense matrix
      __syncthreads();
      for (int b = tid >> 5; b < n_xb; b += NW) expand_batch(b);
    }
  }
  if (tid == 0 && atomicAdd(sched + 1, 1ull) == (unsigned long long)gridDim.x - 1) { sched[0] = 0; sched[1] = 0; }
}

template <int S> int launch_source_S(const DevMech& m, const LaunchCfg& cfg, int mode, int64_t n, int64_t tile,
                                     const double* phi, const double* param, double* out, cudaStream_t st) {
  const int64_t blocks = (n + S - 1) / S;
  source_kernel<S><<<(unsigned)blocks, NT, cfg.smem, st>>>(m, mode, n, tile, phi, param, out);
  return (int)cudaGetLastError();
}
template <int S> int launch_jac_S(const DevMech& m, const DevPlan& p, const LaunchCfg& cfg, int mode, int64_t n, int64_t tile,
                                  const double* phi, const double* param, double* out, unsigned long long* sched, cudaStream_t st) {
  const int64_t tiles = (n + S - 1) / S;
  if (tiles == 0) return 0;
  // persistent grid: as many CTAs as are resident at once (one per SM with 512 threads x 128 registers)
  int dev = 0, n_sm = 0, occ = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e == cudaSuccess) e = cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev);
  const bool expand = p.scratch != nullptr;
  if constexpr (S == 1) {
    if (expand) {                                 // dense by expansion: one CTA per SM, two scratch buffers per CTA
      if (e != cudaSuccess) return (int)e;
      jacobian_kernel<1, 2><<<(unsigned)std::min<int64_t>(tiles, n_sm), NT, cfg.smem, st>>>(m, p, mode, n, tile, phi, param, out, sched);
      return (int)cudaGetLastError();
    }
  }
  if (e == cudaSuccess)
    e = p.nzmask != nullptr ? cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, jacobian_kernel<S, 1>, NT, cfg.smem)
                            : cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, jacobian_kernel<S, 0>, NT, cfg.smem);
  if (e != cudaSuccess) return (int)e;
  const int64_t blocks = std::min<int64_t>(tiles, (int64_t)n_sm * (occ > 0 ? occ : 1));
  if (p.nzmask != nullptr) jacobian_kernel<S, 1><<<(unsigned)blocks, NT, cfg.smem, st>>>(m, p, mode, n, tile, phi, param, out, sched);
  else jacobian_kernel<S, 0><<<(unsigned)blocks, NT, cfg.smem, st>>>(m, p, mode, n, tile, phi, param, out, sched);
  return (int)cudaGetLastError();
}

template <int S> int launch_fd_S(const DevMech& m, const LaunchCfg& cfg, int mode, int ofmt, double rel, double ab, int64_t n,
                                 int64_t tile, int64_t n_e, const double* phi, const double* param, double* out, cudaStream_t st) {
  fd_kernel<S><<<(unsigned)n, NT, cfg.smem, st>>>(m, mode, ofmt, rel, ab, tile, n_e, phi, param, out);
  return (int)cudaGetLastError();
}


}  // namespace

LaunchCfg choose_cfg(const HostTables& h, bool jac, int64_t tile, int64_t n_states, int n_sm) {
  LaunchCfg cfg{1, NT, 0};
  for (int S = 32; S >= 1; S >>= 1) {
    const size_t bytes = smem_doubles(h.ns, h.nr, h.nslots, jac ? h.n_part_jac : h.n_part_src, jac ? h.jplan.n_sg + h.cplan.n_sg : h.qplan.n_sg, S, jac) * sizeof(double);
    cfg.S = S; cfg.smem = bytes;
    if (bytes > SMEM_LIMIT) continue;
    if ((int64_t)S > tile) continue;                       // lanes of one item must stay inside one tile
    if (S > 1 && (n_states + S - 1) / S < 2 * (int64_t)n_sm) continue;  // small batches: spread over the SMs first
    break;
  }
  return cfg;
}

// finite differences: S = columns per pass; the largest that fits, but no wider than the n_var + 1 evaluations
LaunchCfg choose_cfg_fd(const HostTables& h) {
  LaunchCfg cfg{1, NT, 0};
  for (int S = 32; S >= 1; S >>= 1) {
    const size_t bytes = (smem_doubles(h.ns, h.nr, h.nslots, h.n_part_src, h.qplan.n_sg, S, false) + (size_t)h.nvar * (S + 1)) * sizeof(double);
    cfg.S = S; cfg.smem = bytes;
    if (bytes > SMEM_LIMIT) continue;
    if (S > 1 && S / 2 >= h.nvar + 1) continue;
    break;
  }
  return cfg;
}

int launch_fd(const DevMech& m, const LaunchCfg& cfg, int mode, int ofmt, int64_t n_e, double rel_step, double abs_step,
              int64_t n_states, int64_t ld, int64_t tile, const double* phi, const double* param, double* out, void* stream) {
  (void)ld;
  cudaStream_t st = (cudaStream_t)stream;
#define FD_CASE(S_) case S_: return launch_fd_S<S_>(m, cfg, mode, ofmt, rel_step, abs_step, n_states, tile, n_e, phi, param, out, st);
  switch (cfg.S) {
    FD_CASE(1) FD_CASE(2) FD_CASE(4) FD_CASE(8) FD_CASE(16)
    default: return launch_fd_S<32>(m, cfg, mode, ofmt, rel_step, abs_step, n_states, tile, n_e, phi, param, out, st);
  }
#undef FD_CASE
}

int launch_source(const DevMech& m, const LaunchCfg& cfg, int mode, int64_t n_states, int64_t ld, int64_t tile,
                  const double* phi, const double* param, double* out, void* stream) {
  (void)ld;
  cudaStream_t st = (cudaStream_t)stream;
  switch (cfg.S) {
    case 1: return launch_source_S<1>(m, cfg, mode, n_states, tile, phi, param, out, st);
    case 2: return launch_source_S<2>(m, cfg, mode, n_states, tile, phi, param, out, st);
    case 4: return launch_source_S<4>(m, cfg, mode, n_states, tile, phi, param, out, st);
    case 8: return launch_source_S<8>(m, cfg, mode, n_states, tile, phi, param, out, st);
    case 16: return launch_source_S<16>(m, cfg, mode, n_states, tile, phi, param, out, st);
    default: return launch_source_S<32>(m, cfg, mode, n_states, tile, phi, param, out, st);
  }
}

int launch_jacobian(const DevMech& m, const DevPlan& p, const LaunchCfg& cfg, int mode, int64_t n_states, int64_t ld,
                    int64_t tile, const double* phi, const double* param, double* out, unsigned long long* sched, void* stream) {
  (void)ld;
  cudaStream_t st = (cudaStream_t)stream;
  switch (cfg.S) {
    case 1: return launch_jac_S<1>(m, p, cfg, mode, n_states, tile, phi, param, out, sched, st);
    case 2: return launch_jac_S<2>(m, p, cfg, mode, n_states, tile, phi, param, out, sched, st);
    case 4: return launch_jac_S<4>(m, p, cfg, mode, n_states, tile, phi, param, out, sched, st);
    case 8: return launch_jac_S<8>(m, p, cfg, mode, n_states, tile, phi, param, out, sched, st);
    case 16: return launch_jac_S<16>(m, p, cfg, mode, n_states, tile, phi, param, out, sched, st);
    default: return launch_jac_S<32>(m, p, cfg, mode, n_states, tile, phi, param, out, sched, st);
  }
}

template <int S> static int set_attr_S() {
  cudaError_t e = cudaFuncSetAttribute(source_kernel<S>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SMEM_LIMIT);
  if (e != cudaSuccess) return (int)e;
  e = cudaFuncSetAttribute(fd_kernel<S>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SMEM_LIMIT);
  if (e != cudaSuccess) return (int)e;
  e = cudaFuncSetAttribute(jacobian_kernel<S, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SMEM_LIMIT);
  if (e != cudaSuccess) return (int)e;
  if constexpr (S == 1) {
    e = cudaFuncSetAttribute(jacobian_kernel<1, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SMEM_LIMIT);
    if (e != cudaSuccess) return (int)e;
  }
  return (int)cudaFuncSetAttribute(jacobian_kernel<S, 0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SMEM_LIMIT);
}

int set_kernel_attributes() {
  int e;
  if ((e = set_attr_S<1>())) return e;
  if ((e = set_attr_S<2>())) return e;
  if ((e = set_attr_S<4>())) return e;
  if ((e = set_attr_S<8>())) return e;
  if ((e = set_attr_S<16>())) return e;
  return set_attr_S<32>();
}

}  // namespace pyjac
