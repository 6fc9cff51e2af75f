// Step a0 of the hot path (one-time, host): mechanism description -> packed tables, sparsity
// pattern and static gather maps.  The paper bakes this information into generated code
// and searches the CRS/CCS index arrays at run time; here the
// kernels are mechanism-agnostic and read tables, and the run-time search is replaced by static
// maps, as the paper itself proposes.
#include <algorithm>
#include <array>
#include <functional>
#include <cmath>
#include <cstring>
#include <map>
#include <numeric>
#include <sstream>

#include "pyjac_internal.h"

namespace pyjac {

namespace {

struct Role { int species; int slot; };   // a Jacobian slot holding  dQ_i/dC_species  (one role)

#define MECH_FAIL(msg) do { std::ostringstream os_; os_ << msg; err = os_.str(); return PYJAC_EMECH; } while (0)

int validate(const pyjac_mech_desc* d, std::string& err) {
  const int ns = d->n_species, nr = d->n_reactions;
  if (ns < 2) MECH_FAIL("n_species must be >= 2, got " << ns);
  if (nr < 1) MECH_FAIL("n_reactions must be >= 1, got " << nr);
  if (ns > 32767) MECH_FAIL("n_species > 32767 unsupported");
  if (!d->mol_weight || !d->nasa_tmid || !d->nasa_lo || !d->nasa_hi || !d->reac_ptr || !d->reac_species || !d->reac_nu || !d->prod_ptr ||
      !d->prod_species || !d->prod_nu || !d->reversible || !d->type || !d->A || !d->beta || !d->Ta || !d->eff_ptr || !d->collider)
    MECH_FAIL("a required array of the mechanism description is NULL");
  for (int i = 0; i < nr; ++i) {
    if (d->reac_ptr[i + 1] < d->reac_ptr[i] || d->prod_ptr[i + 1] < d->prod_ptr[i] || d->eff_ptr[i + 1] < d->eff_ptr[i])
      MECH_FAIL("reaction " << i << ": pointer arrays must be non-decreasing");
    if (d->eff_ptr[i + 1] > d->eff_ptr[i] && (!d->eff_species || !d->eff_value)) MECH_FAIL("efficiency arrays are NULL");
  }
  for (int k = 0; k < ns; ++k) {
    if (!(d->mol_weight[k] > 0.0)) MECH_FAIL("species " << k << ": molecular weight must be > 0");
    if (!(d->nasa_tmid[k] > 0.0)) MECH_FAIL("species " << k << ": T_mid must be > 0");
  }
  for (int i = 0; i < nr; ++i) {
    const int ty = d->type[i];
    if (ty < PYJAC_ELEMENTARY || ty > PYJAC_CHEBYSHEV) MECH_FAIL("reaction " << i << ": unknown type " << ty);
    for (int side = 0; side < 2; ++side) {
      const int32_t* ptr = side ? d->prod_ptr : d->reac_ptr;
      const int32_t* sp = side ? d->prod_species : d->reac_species;
      const int32_t* nu = side ? d->prod_nu : d->reac_nu;
      const int n = ptr[i + 1] - ptr[i];
      if (n < 1 || n > 3) MECH_FAIL("reaction " << i << ": " << (side ? "products" : "reactants") << " must have 1..3 species, got " << n);
      for (int j = ptr[i]; j < ptr[i + 1]; ++j) {
        if (sp[j] < 0 || sp[j] >= ns) MECH_FAIL("reaction " << i << ": species index " << sp[j] << " out of range");
        if (nu[j] < 1 || nu[j] > 3) MECH_FAIL("reaction " << i << ": stoichiometric coefficient " << nu[j] << " outside 1..3");
        for (int l = ptr[i]; l < j; ++l)
          if (sp[l] == sp[j]) MECH_FAIL("reaction " << i << ": species " << sp[j] << " listed twice on one side");
      }
    }
    {
      int snu = 0;
      for (int j = d->reac_ptr[i]; j < d->reac_ptr[i + 1]; ++j) snu -= d->reac_nu[j];
      for (int j = d->prod_ptr[i]; j < d->prod_ptr[i + 1]; ++j) snu += d->prod_nu[j];
      if (snu < -7 || snu > 7) MECH_FAIL("reaction " << i << ": |sum of stoichiometric coefficients| = " << (snu < 0 ? -snu : snu) << " exceeds 7");
    }
    if (ty >= PYJAC_FALLOFF_LINDEMANN && ty <= PYJAC_FALLOFF_SRI && (!d->low_A || !d->low_beta || !d->low_Ta)) MECH_FAIL("reaction " << i << ": falloff arrays are NULL");
    if (ty == PYJAC_FALLOFF_TROE && (!d->troe || !d->troe_has_T2)) MECH_FAIL("reaction " << i << ": Troe arrays are NULL");
    if (ty == PYJAC_FALLOFF_SRI && !d->sri) MECH_FAIL("reaction " << i << ": SRI array is NULL");
    if (ty == PYJAC_PLOG && (!d->plog_ptr || !d->plog_P || !d->plog_A || !d->plog_beta || !d->plog_Ta)) MECH_FAIL("reaction " << i << ": P-Log arrays are NULL");
    if (ty == PYJAC_CHEBYSHEV && (!d->cheb_ptr || !d->cheb_nT || !d->cheb_nP || !d->cheb_Tmin || !d->cheb_Tmax || !d->cheb_Pmin || !d->cheb_Pmax || !d->cheb_coef))
      MECH_FAIL("reaction " << i << ": Chebyshev arrays are NULL");
    if (ty <= PYJAC_FALLOFF_SRI && !(d->A[i] > 0.0)) MECH_FAIL("reaction " << i << ": A must be > 0 (ln A is tabulated)");
    if (d->chem_activated && d->chem_activated[i] && !(ty >= PYJAC_FALLOFF_LINDEMANN && ty <= PYJAC_FALLOFF_SRI))
      MECH_FAIL("reaction " << i << ": chem_activated needs a falloff type");
    if (d->rev_A && d->rev_A[i] != 0.0) {
      if (!(d->rev_A[i] > 0.0) || !d->rev_beta || !d->rev_Ta) MECH_FAIL("reaction " << i << ": explicit reverse parameters need rev_A > 0, rev_beta and rev_Ta");
      if (!d->reversible[i] || ty == PYJAC_PLOG || ty == PYJAC_CHEBYSHEV)
        MECH_FAIL("reaction " << i << ": explicit reverse parameters need a reversible reaction that is not P-Log / Chebyshev");
    }
    if (ty >= PYJAC_FALLOFF_LINDEMANN && ty <= PYJAC_FALLOFF_SRI && !(d->low_A[i] > 0.0))
      MECH_FAIL("reaction " << i << ": low-pressure A must be > 0");
    if (d->collider[i] < -1 || d->collider[i] >= ns) MECH_FAIL("reaction " << i << ": collider index out of range");
    for (int j = d->eff_ptr[i]; j < d->eff_ptr[i + 1]; ++j) {
      if (d->eff_species[j] < 0 || d->eff_species[j] >= ns) MECH_FAIL("reaction " << i << ": efficiency species out of range");
      if (!(d->eff_value[j] >= 0.0)) MECH_FAIL("reaction " << i << ": negative third-body efficiency");
    }
    if (ty == PYJAC_PLOG) {
      const int n = d->plog_ptr[i + 1] - d->plog_ptr[i];
      int levels = 0;
      for (int j = d->plog_ptr[i]; j < d->plog_ptr[i + 1]; ++j) {
        if (!(d->plog_P[j] > 0.0) || !(d->plog_A[j] > 0.0)) MECH_FAIL("reaction " << i << ": P-Log P and A must be > 0");
        if (j > d->plog_ptr[i] && !(d->plog_P[j] >= d->plog_P[j - 1])) MECH_FAIL("reaction " << i << ": P-Log pressures must be ascending");
        if (j == d->plog_ptr[i] || d->plog_P[j] != d->plog_P[j - 1]) ++levels;      // equal pressures: one level, rates summed (R10)
      }
      if (n < 2 || levels < 2) MECH_FAIL("reaction " << i << ": P-Log needs >= 2 distinct pressures");
    }
    if (ty == PYJAC_CHEBYSHEV) {
      if (d->cheb_nT[i] < 1 || d->cheb_nP[i] < 1) MECH_FAIL("reaction " << i << ": empty Chebyshev grid");
      if (!(d->cheb_Tmin[i] > 0.0) || !(d->cheb_Tmin[i] < d->cheb_Tmax[i])) MECH_FAIL("reaction " << i << ": Chebyshev needs 0 < Tmin < Tmax");
      if (!(d->cheb_Pmin[i] > 0.0) || !(d->cheb_Pmin[i] < d->cheb_Pmax[i])) MECH_FAIL("reaction " << i << ": Chebyshev needs 0 < Pmin < Pmax");
    }
  }
  return PYJAC_OK;
}


// Gather plan.  Every list is cut into segments of at most SEG entries; the segments,
// sorted by DESCENDING length, are packed in ELL "super-groups" of ELL_W segments, padded (with entries pointing at
// an always-zero slot) to the longest segment of the group and stored entry-major: the 32 lanes of a warp read 32
// consecutive entries and a thread keeps several independent loads in flight.  A list that fits one segment is
// stored straight to the output; the segments of a split list leave partial sums in shared memory which a short
// second pass combines.  stride = ints per entry.
// One-word entries (stride 1) are stored PACKED: two consecutive entries of a segment (steps 2q and 2q + 1) in one
// 32-bit word, 15 bits of slot index and a sign bit each -- half the plan traffic and half the entry loads of the
// gathers.  The slots live in shared memory as doubles (<= 227 KB), so an index always fits 15 bits for a mechanism the
// tile kernels can run; `packable` = false otherwise (the plan is then left unpacked and must not be used by them).
void build_gather(const std::vector<std::vector<int32_t>>& lists, int stride, int zero_slot, int narrow_len, GatherPlan& g) {
  const int SEG = SEG_LEN;
  const int n = (int)lists.size();
  g = GatherPlan();
  g.stride = stride;
  g.packed = stride == 1;
  if (g.packed) {
    g.packable = zero_slot + N_ZERO_SLOTS <= 0x8000;
    for (const auto& l : lists) for (int32_t e : l) g.packable &= ((uint32_t)e & ~SIGN_BIT) < 0x8000u;
    g.packed = g.packable;
  }
  struct Seg { int item, p0, len, target; };
  std::vector<Seg> segs;
  for (int i = 0; i < n; ++i) {
    const int len = (int)lists[i].size() / stride;
    g.n_entries += len;
    if (len <= SEG) { segs.push_back({i, 0, len, i}); continue; }
    const int nseg = (len + SEG - 1) / SEG;
    g.comb_item.push_back(i); g.comb_first.push_back(g.n_part); g.comb_nseg.push_back(nseg);
    for (int q = 0; q < nseg; ++q) {               // nearly equal pieces
      const int a = (int)((int64_t)len * q / nseg), b = (int)((int64_t)len * (q + 1) / nseg);
      segs.push_back({i, a, b - a, -2 - g.n_part++});
    }
  }
  // pieces of split lists (their sums go to shared memory) never join the narrow tail: its store path has no such case
  auto eff_len = [&](const Seg& a) { return a.target <= -2 ? std::max(a.len, narrow_len + 1) : a.len; };
  std::stable_sort(segs.begin(), segs.end(), [&](const Seg& a, const Seg& b) { return eff_len(a) > eff_len(b); });
  const int ns_ = (int)segs.size();
  // Wide super-groups of ELL_W segments first; the tail of short segments (<= narrow_len entries) goes into NARROW
  // super-groups of ELL_W_NARROW segments: a thread then owns 4x as many segments of a unit, so the fixed cost of a
  // unit (work counter, metadata, one exposed round trip for the first entries) is paid a quarter as often.
  int i_n = ns_;
  for (int i = 0; i < ns_; ++i) if (eff_len(segs[i]) <= narrow_len) { i_n = i; break; }
  g.n_wide = (i_n + ELL_W - 1) / ELL_W;
  // plans whose kernels walk wide groups only (narrow_len == 0: T/E rows, source terms) get no narrow groups, however
  // many empty lists there are (inert species still need their stores)
  if (narrow_len == 0) g.n_wide = (ns_ + ELL_W - 1) / ELL_W;
  const int rest = std::max(0, ns_ - g.n_wide * ELL_W);
  g.n_sg = g.n_wide + (rest + ELL_W_NARROW - 1) / ELL_W_NARROW;
  auto group_first = [&](int sg) { return sg < g.n_wide ? sg * ELL_W : g.n_wide * ELL_W + (sg - g.n_wide) * ELL_W_NARROW; };
  auto group_size = [&](int sg) { return sg < g.n_wide ? ELL_W : ELL_W_NARROW; };
  // Shared-memory banks.  At step p the 16 lanes of a half-warp read the p-th entries of 16 consecutive segments,
  // one 8-byte slot each (S = 1; with S states per item the half-warp covers 16/S segments and needs distinct slots
  // mod 16/S, which distinct mod 16 implies).  The order of the entries inside a segment is free, so every block of
  // 16 segments is scheduled step by step with a maximum bipartite matching lanes <-> banks (slot mod 16); padding
  // entries take whichever of the N_ZERO_SLOTS always-zero slots falls in a free bank.
  std::vector<std::vector<int>> order(ns_);           // per sorted segment: entry indices in issue order
  for (int b0 = 0; b0 < ns_; b0 += 16) {
    const int nb = std::min(16, ns_ - b0);
    std::vector<std::vector<int>> rem(nb);
    for (int l = 0; l < nb; ++l) for (int e = 0; e < segs[b0 + l].len; ++e) rem[l].push_back(segs[b0 + l].p0 + e);
    auto bank_of = [&](int l, int e) { return (int)((uint32_t)lists[segs[b0 + l].item][(size_t)e * stride] & ~SIGN_BIT) & 15; };
    for (;;) {
      bool any = false;
      for (int l = 0; l < nb; ++l) any |= !rem[l].empty();
      if (!any) break;
      int owner[16]; std::fill(owner, owner + 16, -1);            // bank -> lane
      std::function<bool(int, uint32_t&)> augment = [&](int l, uint32_t& seen) -> bool {
        for (int e : rem[l]) {
          const int bk = bank_of(l, e);
          if (seen >> bk & 1) continue;
          seen |= 1u << bk;
          if (owner[bk] < 0 || augment(owner[bk], seen)) { owner[bk] = l; return true; }
        }
        return false;
      };
      // longest remaining lists first: they have the fewest later chances to dodge a conflict
      std::vector<int> lanes;
      for (int l = 0; l < nb; ++l) if (!rem[l].empty()) lanes.push_back(l);
      std::stable_sort(lanes.begin(), lanes.end(), [&](int a, int b) { return rem[a].size() > rem[b].size(); });
      for (int l : lanes) { uint32_t seen = 0; augment(l, seen); }
      int pick[16]; std::fill(pick, pick + 16, -1);
      for (int bk = 0; bk < 16; ++bk) if (owner[bk] >= 0) pick[owner[bk]] = bk;
      for (int l : lanes) {
        size_t at = 0;
        if (pick[l] >= 0) for (size_t q = 0; q < rem[l].size(); ++q) if (bank_of(l, rem[l][q]) == pick[l]) { at = q; break; }
        order[b0 + l].push_back(rem[l][at]);
        rem[l].erase(rem[l].begin() + at);
      }
    }
  }
  int off = 0;
  for (int sg = 0; sg < g.n_sg; ++sg) {
    const int i0 = group_first(sg), EW = group_size(sg);
    int width = 0;                                    // the longest segment of the group
    for (int w = 0; w < EW && i0 + w < ns_; ++w) width = std::max(width, segs[i0 + w].len);
    if (g.packed) width = (width + 1) & ~1;           // whole words
    g.sg_meta.push_back(off); g.sg_meta.push_back(g.packed ? width / 2 : width);
    const size_t first_ent = g.ell_ent.size();
    for (int p = 0; p < width; ++p)
      for (int w0 = 0; w0 < EW; w0 += 16) {
        uint32_t used = 0;                            // banks taken by the real entries of this half-warp step
        for (int w = w0; w < w0 + 16; ++w)
          if (i0 + w < ns_ && p < segs[i0 + w].len)
            used |= 1u << (((uint32_t)lists[segs[i0 + w].item][(size_t)order[i0 + w][p] * stride] & ~SIGN_BIT) & 15);
        for (int w = w0; w < w0 + 16; ++w) {
          const bool real = i0 + w < ns_ && p < segs[i0 + w].len;
          int zs = zero_slot;
          if (!real) {                                // a zero slot in a free bank, if one is left
            for (int z = 0; z < N_ZERO_SLOTS; ++z) if (!(used >> ((zero_slot + z) & 15) & 1)) { zs = zero_slot + z; used |= 1u << (zs & 15); break; }
          }
          for (int c = 0; c < stride; ++c)
            g.ell_ent.push_back(real ? lists[segs[i0 + w].item][(size_t)order[i0 + w][p] * stride + c] : (c == 0 ? zs : 0));
        }
      }
    if (g.packed) {                                   // rows 2q and 2q + 1 -> one row of words
      auto half = [](int32_t e) { return ((uint32_t)e & 0x7fffu) | (((uint32_t)e & SIGN_BIT) ? 0x8000u : 0u); };
      std::vector<int32_t> rows(g.ell_ent.begin() + first_ent, g.ell_ent.end());
      g.ell_ent.resize(first_ent);
      for (int q = 0; q < width / 2; ++q)
        for (int w = 0; w < EW; ++w)
          g.ell_ent.push_back((int32_t)(half(rows[(size_t)(2 * q) * EW + w]) | (half(rows[(size_t)(2 * q + 1) * EW + w]) << 16)));
      off += width / 2 * EW;
    } else {
      off += width * EW;
    }
    for (int w = 0; w < EW; ++w) g.target.push_back(i0 + w < ns_ ? segs[i0 + w].target : -1);
  }
  g.n_padded = off;
}

}  // namespace

int build_host_tables(const pyjac_mech_desc* d, bool approx, HostTables& h, std::string& err) {
  if (int rc = validate(d, err)) return rc;
  const int ns = d->n_species, nr = d->n_reactions, nvar = ns + 1, L = ns - 1;
  h.ns = ns; h.nr = nr; h.nvar = nvar;

  // ---- species tables ---------------------------------------------------------------------------
  h.nasa.assign((size_t)ns * 15, 0.0);                 // coefficient-major: [0] tmid, [1..7] low range, [8..14] high range
  h.wr.resize(ns);
  for (int k = 0; k < ns; ++k) {
    h.nasa[k] = d->nasa_tmid[k];
    for (int j = 0; j < 7; ++j) { h.nasa[(size_t)(1 + j) * ns + k] = d->nasa_lo[7 * k + j]; h.nasa[(size_t)(8 + j) * ns + k] = d->nasa_hi[7 * k + j]; }
    h.wr[k] = d->mol_weight[k] / d->mol_weight[L];
  }

  // ---- sort reactions by DESCENDING cost class (type, reversible, non-unit coefficients): warps become
  // type-uniform (the paper's reaction-sorting idea) and the expensive falloff / P-Log / Chebyshev
  // reactions are started first (the kernel hands out 32-reaction chunks dynamically) ---------------------------
  // fast path of the reaction phase (INFO_FAST): most reactions of a real mechanism
  auto is_fast = [&](int i) {
    const int ty = d->type[i];
    if (ty != PYJAC_ELEMENTARY && ty != PYJAC_THIRD_BODY) return false;
    if (d->rev_A && d->rev_A[i] > 0.0) return false;
    const int nre = d->reac_ptr[i + 1] - d->reac_ptr[i], npr = d->prod_ptr[i + 1] - d->prod_ptr[i];
    if (nre > 2 || npr > 2) return false;
    for (int j = d->reac_ptr[i]; j < d->reac_ptr[i + 1]; ++j) if (d->reac_nu[j] != 1 || d->reac_species[j] == L) return false;
    for (int j = d->prod_ptr[i]; j < d->prod_ptr[i + 1]; ++j) if (d->prod_nu[j] != 1 || (d->reversible[i] && d->prod_species[j] == L)) return false;
    if (ty == PYJAC_THIRD_BODY) {
      if (d->collider[i] == L) return false;
      for (int j = d->eff_ptr[i]; j < d->eff_ptr[i + 1]; ++j) if (d->eff_species[j] == L && d->eff_value[j] != 1.0) return false;
    }
    return true;
  };
  h.perm.resize(nr);
  std::iota(h.perm.begin(), h.perm.end(), 0);
  std::stable_sort(h.perm.begin(), h.perm.end(), [&](int a, int b) {
    auto simple = [&](int i) {
      for (int j = d->reac_ptr[i]; j < d->reac_ptr[i + 1]; ++j) if (d->reac_nu[j] != 1) return 0;
      for (int j = d->prod_ptr[i]; j < d->prod_ptr[i + 1]; ++j) if (d->prod_nu[j] != 1) return 0;
      return 1;
    };
    auto cost = [&](int i) {
      static const int rank[7] = {0, 1, 2, 5, 4, 3, 6};   // elementary < third body < Lindemann < P-Log < SRI < Troe < Chebyshev
      return rank[d->type[i]] * 4 + (d->reversible[i] ? 2 : 0) + (simple(i) ? 0 : 1) + (is_fast(i) ? 0 : 64);
    };
    return cost(a) > cost(b);
  });
  // ---- shared-memory banks of phase 1.  Lane r % 32 of a warp reads the thermo records (16-byte loads: a
  // quarter-warp = 8 consecutive reactions is conflict-free iff their species at stoichiometric position a differ
  // mod 8) and the concentrations (8-byte loads: half-warp, species distinct mod 16) of its reaction's species.
  // Inside a cost class the order of the reactions is free, and so is the order of the species on a side: both are
  // chosen greedily to keep the species of neighbouring lanes in different banks.
  std::vector<std::array<int, 6>> sp_order(nr);       // [sorted r][position a] -> index into the reactant (a < 3) / product list, -1 unused
  {
    auto cost_class = [&](int i) {
      static const int rank[7] = {0, 1, 2, 5, 4, 3, 6};
      bool simple = true;
      for (int j = d->reac_ptr[i]; j < d->reac_ptr[i + 1]; ++j) simple &= d->reac_nu[j] == 1;
      for (int j = d->prod_ptr[i]; j < d->prod_ptr[i + 1]; ++j) simple &= d->prod_nu[j] == 1;
      return rank[d->type[i]] * 4 + (d->reversible[i] ? 2 : 0) + (simple ? 0 : 1) + (is_fast(i) ? 0 : 64);
    };
    std::vector<std::array<int, 6>> placed(nr);       // species at each position of the reactions placed so far (ns = dummy)
    auto species_at = [&](int i, const std::array<int, 6>& o, int a) {
      if (o[a] < 0) return ns;
      return a < 3 ? d->reac_species[d->reac_ptr[i] + o[a]] : d->prod_species[d->prod_ptr[i] + o[a]];
    };
    auto conflicts = [&](int r, const std::array<int, 6>& spc) {      // against the lanes already placed
      int c = 0;
      for (int q = r - r % 16; q < r; ++q)
        for (int a = 0; a < 6; ++a) {
          if (placed[q][a] == spc[a]) continue;                      // same address: broadcast
          if (q >= r - r % 8 && (placed[q][a] & 7) == (spc[a] & 7)) c += 4;   // two 16-byte loads per species
          if ((placed[q][a] & 15) == (spc[a] & 15)) c += 1;
        }
      return c;
    };
    int r0 = 0;
    while (r0 < nr) {
      int r1 = r0;
      while (r1 < nr && cost_class(h.perm[r1]) == cost_class(h.perm[r0])) ++r1;
      std::vector<int> pool(h.perm.begin() + r0, h.perm.begin() + r1);
      for (int r = r0; r < r1; ++r) {
        int best = -1, best_c = 1 << 30; std::array<int, 6> best_o{}, best_s{};
        for (size_t c = 0; c < pool.size(); ++c) {
          const int i = pool[c];
          const int nre = d->reac_ptr[i + 1] - d->reac_ptr[i], npr = d->prod_ptr[i + 1] - d->prod_ptr[i];
          for (int sw = 0; sw < 4; ++sw) {                           // swap the first two reactants / products
            if ((sw & 1) && nre < 2) continue;
            if ((sw & 2) && npr < 2) continue;
            std::array<int, 6> o = {nre > 0 ? 0 : -1, nre > 1 ? 1 : -1, nre > 2 ? 2 : -1, npr > 0 ? 0 : -1, npr > 1 ? 1 : -1, npr > 2 ? 2 : -1};
            if (sw & 1) std::swap(o[0], o[1]);
            if (sw & 2) std::swap(o[3], o[4]);
            std::array<int, 6> spc;
            for (int a = 0; a < 6; ++a) spc[a] = species_at(i, o, a);
            const int cc = conflicts(r, spc);
            if (cc < best_c) { best_c = cc; best = (int)c; best_o = o; best_s = spc; }
          }
          if (best_c == 0) break;
        }
        h.perm[r] = pool[best]; sp_order[r] = best_o; placed[r] = best_s;
        pool.erase(pool.begin() + best);
      }
      r0 = r1;
    }
  }

  // ---- reaction chunks of phase 1: a new chunk wherever the cost group changes ----------------------------------
  for (int ls = 0; ls < 6; ++ls) {
    static const int rank[7] = {0, 1, 2, 5, 4, 3, 6};
    auto group = [&](int r) { const int i = h.perm[r]; return is_fast(i) ? 100 : rank[d->type[i]]; };
    const int cap = 32 >> ls;
    h.rxc[ls].clear();
    for (int r = 0; r < nr;) {
      int e = r + 1;
      while (e < nr && e - r < cap && group(e) == group(r)) ++e;
      h.rxc[ls].push_back(r); h.rxc[ls].push_back(e);
      r = e;
    }
  }

  h.lnA.resize(nr); h.beta.resize(nr); h.Ta.resize(nr); h.dn.resize(nr);
  h.info.resize(nr); h.aux.assign(nr, -1); h.sp.assign((size_t)nr * 8, (uint32_t)ns);
  h.eff_ptr.assign(1, 0); h.slot_base.assign(1, 0);
  std::vector<std::vector<Role>> roles(nr);
  std::vector<std::vector<std::pair<int, int>>> net(nr);   // (species k < Ns-1... incl. last, net nu != 0)

  for (int r = 0; r < nr; ++r) {
    const int i = h.perm[r];
    const int ty = d->type[i];
    const bool rev = d->reversible[i] != 0;
    const bool tb = ty >= PYJAC_THIRD_BODY && ty <= PYJAC_FALLOFF_SRI;
    const bool falloff = ty >= PYJAC_FALLOFF_LINDEMANN && ty <= PYJAC_FALLOFF_SRI;
    // chemically activated (R8): the rate constant of the rates of progress is k_0, so the Arrhenius
    // columns take the LOW parameters and the falloff record the high-pressure ones (the kernel inverts the ratio)
    const bool chem = falloff && d->chem_activated && d->chem_activated[i];
    h.lnA[r] = (ty <= PYJAC_FALLOFF_SRI) ? std::log(chem ? d->low_A[i] : d->A[i]) : 0.0;
    h.beta[r] = chem ? d->low_beta[i] : d->beta[i]; h.Ta[r] = chem ? d->low_Ta[i] : d->Ta[i];
    const int nre = d->reac_ptr[i + 1] - d->reac_ptr[i], npr = d->prod_ptr[i + 1] - d->prod_ptr[i];
    int snu = 0, order_f = 0, order_r = 0;
    bool simple = true;
    std::map<int, int> netnu;
    for (int a = 0; a < nre; ++a) {
      const int j = d->reac_ptr[i] + sp_order[r][a];
      h.sp[8 * r + a] = (uint32_t)d->reac_species[j] | ((uint32_t)d->reac_nu[j] << 16);
      snu -= d->reac_nu[j]; netnu[d->reac_species[j]] -= d->reac_nu[j];
      order_f += d->reac_nu[j]; simple &= d->reac_nu[j] == 1;
    }
    for (int b = 0; b < npr; ++b) {
      const int j = d->prod_ptr[i] + sp_order[r][3 + b];
      h.sp[8 * r + 3 + b] = (uint32_t)d->prod_species[j] | ((uint32_t)d->prod_nu[j] << 16);
      snu += d->prod_nu[j]; netnu[d->prod_species[j]] += d->prod_nu[j];
      order_r += d->prod_nu[j]; simple &= d->prod_nu[j] == 1;
    }
    double dn = 0.0;
    for (auto& kv : netnu)
      if (kv.second != 0) { net[r].push_back(kv); if (kv.first != L) dn += kv.second * (1.0 - h.wr[kv.first]); }
    h.dn[r] = dn;
    const bool adef = tb && d->collider[i] < 0;
    int info = ty | (rev ? INFO_REV : 0) | (adef ? INFO_ADEF : 0) | ((snu + 8) << INFO_SNU_SHIFT) |
               (nre << INFO_NREAC_SHIFT) | (npr << INFO_NPROD_SHIFT) | (simple ? INFO_SIMPLE : 0) |
               (order_f << INFO_OF_SHIFT) | (order_r << INFO_OR_SHIFT);
    if (ty == PYJAC_FALLOFF_TROE && d->troe_has_T2[i]) info |= INFO_T2;
    if (chem) info |= INFO_CHEM;
    if (is_fast(i)) info |= INFO_FAST;
    if (rev && d->rev_A && d->rev_A[i] > 0.0) {
      info |= INFO_REVX;
      if (h.rev_par.empty()) h.rev_par.assign((size_t)nr * 3, 0.0);
      h.rev_par[3 * r] = std::log(d->rev_A[i]); h.rev_par[3 * r + 1] = d->rev_beta[i]; h.rev_par[3 * r + 2] = d->rev_Ta[i];
    }
    h.info[r] = info;
    // slots: 0 = T column, 1 = E column, then one per role
    int slot = h.slot_base[r] + 2;
    for (int a = 0; a < nre; ++a) roles[r].push_back({d->reac_species[d->reac_ptr[i] + sp_order[r][a]], slot++});
    if (rev) for (int b = 0; b < npr; ++b) roles[r].push_back({d->prod_species[d->prod_ptr[i] + sp_order[r][3 + b]], slot++});
    if (tb) {
      if (d->collider[i] >= 0) {           // [M] = C_collider: default 0, one efficiency of 1
        h.eff_sp.push_back(d->collider[i]); h.eff_d.push_back(1.0);
        roles[r].push_back({d->collider[i], slot++});
      } else {
        for (int j = d->eff_ptr[i]; j < d->eff_ptr[i + 1]; ++j) {
          if (d->eff_value[j] == 1.0) continue;
          bool dup = false;
          for (int l = d->eff_ptr[i]; l < j; ++l) dup |= d->eff_species[l] == d->eff_species[j];
          if (dup) MECH_FAIL("reaction " << i << ": efficiency of species " << d->eff_species[j] << " given twice");
          h.eff_sp.push_back(d->eff_species[j]); h.eff_d.push_back(d->eff_value[j] - 1.0);
          roles[r].push_back({d->eff_species[j], slot++});
        }
      }
    }
    h.eff_ptr.push_back((int)h.eff_sp.size());
    h.max_eff = std::max(h.max_eff, h.eff_ptr[r + 1] - h.eff_ptr[r]);
    h.slot_base.push_back(slot);
    if (falloff) {
      h.aux[r] = (int)(h.fall.size() / 12);
      double f[12] = {std::log(chem ? d->A[i] : d->low_A[i]), chem ? d->beta[i] : d->low_beta[i], chem ? d->Ta[i] : d->low_Ta[i],
                      0, 0, 0, 0, 0, 0, 0, 0, 0};
      if (ty == PYJAC_FALLOFF_TROE) for (int j = 0; j < 4; ++j) f[4 + j] = d->troe[4 * i + j];
      if (ty == PYJAC_FALLOFF_SRI) for (int j = 0; j < 5; ++j) f[4 + j] = d->sri[5 * i + j];
      h.fall.insert(h.fall.end(), f, f + 12);
    } else if (ty == PYJAC_PLOG) {
      // pressure LEVELS: entries of equal pressure form one level whose rate is the sum of theirs (R10)
      if (h.plog_ptr.empty()) { h.plog_ptr.push_back(0); h.plog_ent.push_back(0); }
      h.aux[r] = (int)h.plog_ptr.size() - 1;
      for (int j = d->plog_ptr[i]; j < d->plog_ptr[i + 1]; ++j) {
        if (j == d->plog_ptr[i] || d->plog_P[j] != d->plog_P[j - 1]) {
          if (j > d->plog_ptr[i]) h.plog_ent.push_back((int)h.plog_lnA.size());
          h.plog_P.push_back(d->plog_P[j]); h.plog_lnP.push_back(std::log(d->plog_P[j]));
        }
        h.plog_lnA.push_back(std::log(d->plog_A[j])); h.plog_b.push_back(d->plog_beta[j]); h.plog_Ta.push_back(d->plog_Ta[j]);
      }
      h.plog_ent.push_back((int)h.plog_lnA.size());
      h.plog_ptr.push_back((int)h.plog_P.size());
    } else if (ty == PYJAC_CHEBYSHEV) {
      h.aux[r] = (int)(h.cheb_meta.size() / 4);
      const int nT = d->cheb_nT[i], nP = d->cheb_nP[i];
      h.cheb_meta.insert(h.cheb_meta.end(), {nT, nP, (int)h.cheb_coef.size(), 0});
      h.cheb_lim.insert(h.cheb_lim.end(), {1.0 / d->cheb_Tmin[i], 1.0 / d->cheb_Tmax[i], std::log10(d->cheb_Pmin[i]), std::log10(d->cheb_Pmax[i])});
      for (int j = 0; j < nT * nP; ++j) h.cheb_coef.push_back(d->cheb_coef[d->cheb_ptr[i] + j]);
    }
  }
  h.nslots = h.slot_base[nr];

  // ---- gather maps and pattern (R5) ----------------------------------------
  // Species-block entry (k, j), k, j < L:  J = sum_i nu_ki (Ghat^j_i - Ghat^L_i)  (R4-6):
  // + every role of species j, - every role of the last species L (those hit ALL columns: dense rows).
  std::vector<std::map<int, std::vector<int32_t>>> rowmap(L);   // row k -> col j -> entries
  std::vector<std::vector<int32_t>> bl(L), bql(L), cl(L);
  auto push_n = [](std::vector<int32_t>& v, int32_t e, int n) { for (int c = 0; c < n; ++c) v.push_back(e); };
  for (int r = 0; r < nr; ++r) {
    for (auto& kv : net[r]) {
      const int k = kv.first, nu = kv.second;
      if (k == L) continue;
      const uint32_t sgn = nu < 0 ? SIGN_BIT : 0u;
      push_n(bl[k], (int32_t)((uint32_t)h.slot_base[r] | sgn), std::abs(nu));
      push_n(bql[k], (int32_t)((uint32_t)r | sgn), std::abs(nu));
      for (const Role& ro : roles[r]) {
        if (ro.species != L) push_n(rowmap[k][ro.species], (int32_t)((uint32_t)ro.slot | sgn), std::abs(nu));
        else if (!approx)      // exact Jacobian: C_Ns depends on every n_j -> dense row; dropped by the
                               // "approximate" switch of PAPER.md L313-317
          for (int j = 0; j < L; ++j) push_n(rowmap[k][j], (int32_t)((uint32_t)ro.slot | (sgn ^ SIGN_BIT)), std::abs(nu));
      }
    }
    if (!net[r].empty() && !(net[r].size() == 1 && net[r][0].first == L)) {
      for (const Role& ro : roles[r]) {
        if (ro.species != L) { cl[ro.species].push_back(ro.slot); cl[ro.species].push_back(r); }
        else if (!approx) for (int j = 0; j < L; ++j) { cl[j].push_back((int32_t)((uint32_t)ro.slot | SIGN_BIT)); cl[j].push_back(r); }
      }
    }
  }
  // exact structural pattern by the rule of DESIGN.md R5: a pair (k, j) reached only through terms that
  // cancel identically (alpha_ij == alpha_iL, both non-default) is NOT a structural nonzero.
  {
    std::vector<std::vector<char>> inpat(L, std::vector<char>(L, 0));
    for (int r = 0; r < nr; ++r) {
      const int i = h.perm[r];
      const int ty = d->type[i];
      const bool rev = d->reversible[i] != 0;
      const bool tb = ty >= PYJAC_THIRD_BODY && ty <= PYJAC_FALLOFF_SRI;
      auto dep = [&](int k) {
        for (int j = d->reac_ptr[i]; j < d->reac_ptr[i + 1]; ++j) if (d->reac_species[j] == k) return true;
        if (rev) for (int j = d->prod_ptr[i]; j < d->prod_ptr[i + 1]; ++j) if (d->prod_species[j] == k) return true;
        return false;
      };
      auto alpha = [&](int k) {
        if (d->collider[i] >= 0) return k == d->collider[i] ? 1.0 : 0.0;
        for (int j = d->eff_ptr[i]; j < d->eff_ptr[i + 1]; ++j) if (d->eff_species[j] == k) return d->eff_value[j];
        return 1.0;
      };
      const bool depL = dep(L);
      const double aL = tb ? alpha(L) : 0.0;
      for (auto& kv : net[r]) {
        if (kv.first == L) continue;
        for (int j = 0; j < L; ++j)
          if (approx ? (dep(j) || (tb && alpha(j) != (d->collider[i] >= 0 ? 0.0 : 1.0)))
                     : (depL || dep(j) || (tb && alpha(j) != aL))) inpat[kv.first][j] = 1;
      }
    }
    for (int k = 0; k < L; ++k) {
      for (auto it = rowmap[k].begin(); it != rowmap[k].end();)
        it = inpat[k][it->first] ? std::next(it) : rowmap[k].erase(it);
      for (int j = 0; j < L; ++j)
        if (inpat[k][j] && !rowmap[k].count(j)) MECH_FAIL("internal: pattern entry (" << k << "," << j << ") has no gather list");
    }
  }
  // pattern: rows T, E dense; columns T, E dense (R5 / S10); species block from rowmap
  std::vector<std::vector<int>> rows(nvar);
  for (int r = 0; r < 2; ++r) { rows[r].resize(nvar); std::iota(rows[r].begin(), rows[r].end(), 0); }
  for (int k = 0; k < L; ++k) {
    rows[2 + k] = {0, 1};
    for (auto& kv : rowmap[k]) rows[2 + k].push_back(2 + kv.first);
  }
  h.csr_ptr.assign(1, 0);
  for (int r = 0; r < nvar; ++r) { h.csr_idx.insert(h.csr_idx.end(), rows[r].begin(), rows[r].end()); h.csr_ptr.push_back((int)h.csr_idx.size()); }
  h.nnz = (int64_t)h.csr_idx.size();
  if ((int64_t)nvar * nvar > 2147483647LL) MECH_FAIL("n_var^2 exceeds int32");
  // CSC = transpose; csr2csc[p] = position of CSR entry p in CSC value order
  std::vector<int> colcount(nvar + 1, 0);
  for (int c : h.csr_idx) colcount[c + 1]++;
  h.csc_ptr.assign(nvar + 1, 0);
  for (int c = 0; c < nvar; ++c) h.csc_ptr[c + 1] = h.csc_ptr[c] + colcount[c + 1];
  h.csc_idx.resize(h.nnz);
  std::vector<int> fill(h.csc_ptr.begin(), h.csc_ptr.end() - 1), csr2csc(h.nnz);
  for (int r = 0; r < nvar; ++r)
    for (int p = h.csr_ptr[r]; p < h.csr_ptr[r + 1]; ++p) { const int c = h.csr_idx[p]; csr2csc[p] = fill[c]; h.csc_idx[fill[c]++] = r; }
  // finite-difference kernel: it works column by column, so it walks the CSC pattern and needs the
  // CSR value position of every CSC entry
  h.csc2csr.resize(h.nnz);
  for (int64_t p = 0; p < h.nnz; ++p) h.csc2csr[csr2csc[p]] = (int32_t)p;
  auto csr_pos = [&](int r, int c) {
    auto b = h.csr_idx.begin() + h.csr_ptr[r], e = h.csr_idx.begin() + h.csr_ptr[r + 1];
    return (int)(std::lower_bound(b, e, c) - h.csr_idx.begin());
  };
  auto pos_of = [&](int fmt, int r, int c) -> int32_t {
    switch (fmt) {
      case OUT_CSR: return csr_pos(r, c);
      case OUT_CSC: return csr2csc[csr_pos(r, c)];
      case OUT_DENSE_C: return r * nvar + c;
      default: return c * nvar + r;
    }
  };
  // ---- gather plans ------------------------------------------------------------
  // J-plan items: species-block nonzeros (k, j) in row-major order, then the T and E columns of the species rows.
  struct Item { int r, c; };
  std::vector<Item> jitems;
  std::vector<std::vector<int32_t>> jlists;
  for (int k = 0; k < L; ++k)
    for (auto& kv : rowmap[k]) { jitems.push_back({2 + k, 2 + kv.first}); jlists.push_back(kv.second); }
  h.nA = (int)jitems.size();
  // raw gather lists (old slot numbering) for the block-partitioned plan of the Jacobian kernel (pyjac_plan.cpp)
  h.raw_blk = jlists;
  for (const Item& it : jitems) { h.blk_r.push_back(it.r); h.blk_c.push_back(it.c); }
  h.raw_col = bl;
  h.raw_row = cl;
  h.csr2csc.assign(csr2csc.begin(), csr2csc.end());
  for (int col = 0; col < 2; ++col)
    for (int k = 0; k < L; ++k) {
      std::vector<int32_t> l = bl[k];
      for (auto& e : l) e += col;                      // slot base + 0: T column, + 1: E column (sign bit untouched)
      jitems.push_back({2 + k, col}); jlists.push_back(std::move(l));
    }
  build_gather(jlists, 1, h.nslots, NARROW_LEN, h.jplan);
  std::vector<std::vector<int32_t>> clists(L), qlists(L);
  for (int k = 0; k < L; ++k) {
    qlists[k] = bql[k];
    for (size_t e = 0; e + 1 < cl[k].size(); e += 2) {   // entry = (slot | sign, reaction, dn~ of the reaction as 2 ints)
      int32_t w[2];
      std::memcpy(w, &h.dn[cl[k][e + 1]], 8);
      clists[k].insert(clists[k].end(), {cl[k][e], cl[k][e + 1], w[0], w[1]});
    }
  }
  build_gather(clists, 4, h.nslots, 0, h.cplan);            // T and E rows: (slot | sign, reaction, dn~)
  build_gather(qlists, 1, nr, 0, h.qplan);                  // source terms: omega_k = sum nu_ki q_i
  h.q_target = h.qplan.target;
  h.n_part_jac = h.jplan.n_part + 2 * h.cplan.n_part;
  h.n_part_src = h.qplan.n_part;
  for (int fmt = 0; fmt < 4; ++fmt) {
    h.j_pos[fmt] = h.jplan.target;                     // padding and partial codes stay as they are
    for (size_t e = 0; e < h.jplan.target.size(); ++e)
      if (h.jplan.target[e] >= 0) h.j_pos[fmt][e] = pos_of(fmt, jitems[h.jplan.target[e]].r, jitems[h.jplan.target[e]].c);
    h.jc_pos[fmt].clear();
    for (int it : h.jplan.comb_item) h.jc_pos[fmt].push_back(pos_of(fmt, jitems[it].r, jitems[it].c));
    h.c_pos[fmt].assign(2 * h.cplan.target.size(), -1);
    for (size_t e = 0; e < h.cplan.target.size(); ++e) {
      const int tg = h.cplan.target[e];
      h.c_pos[fmt][2 * e] = tg;
      if (tg >= 0) { h.c_pos[fmt][2 * e] = pos_of(fmt, 0, 2 + tg); h.c_pos[fmt][2 * e + 1] = pos_of(fmt, 1, 2 + tg); }
    }
    h.cc_pos[fmt].clear();
    for (int it : h.cplan.comb_item) { h.cc_pos[fmt].push_back(pos_of(fmt, 0, 2 + it)); h.cc_pos[fmt].push_back(pos_of(fmt, 1, 2 + it)); }
    h.d_pos[fmt][0] = pos_of(fmt, 0, 0); h.d_pos[fmt][1] = pos_of(fmt, 0, 1);
    h.d_pos[fmt][2] = pos_of(fmt, 1, 0); h.d_pos[fmt][3] = pos_of(fmt, 1, 1);
  }
  for (int p = 0; p < 2; ++p) {
    h.nzmask[p].assign(((size_t)nvar * nvar + 31) / 32, 0u);
    for (int r = 0; r < nvar; ++r)
      for (int q = h.csr_ptr[r]; q < h.csr_ptr[r + 1]; ++q) {
        const size_t e = p == 0 ? (size_t)r * nvar + h.csr_idx[q] : (size_t)h.csr_idx[q] * nvar + r;
        h.nzmask[p][e >> 5] |= 1u << (e & 31);
      }
    std::vector<int32_t> rank(h.nzmask[p].size() + 1, 0);       // set bits before every word: the CSR / CSC position
    for (size_t w = 1; w <= h.nzmask[p].size(); ++w) rank[w] = rank[w - 1] + __builtin_popcount(h.nzmask[p][w - 1]);
    const int64_t n2 = (int64_t)h.nvar * h.nvar;
    auto present = [&](int64_t e) { return e >= 0 && e < n2 && ((h.nzmask[p][e >> 5] >> (e & 31)) & 1u); };
    auto rank_of = [&](int64_t e) { return rank[e >> 5] + __builtin_popcount(h.nzmask[p][e >> 5] & ((1u << (e & 31)) - 1u)); };
    for (int sh = 0; sh < 2; ++sh) {
      const int64_t n_pairs = (n2 + sh + 1) / 2;
      std::vector<int32_t>& x = h.xpair[2 * p + sh];
      x.assign((size_t)((n_pairs + XPAIR_PAD - 1) / XPAIR_PAD * XPAIR_PAD), 0);
      for (int64_t q = 0; q < n_pairs; ++q) {
        const int64_t e1 = 2 * q - sh, e2 = e1 + 1;
        const bool b1 = present(e1), b2 = present(e2);
        if (b1 || b2) x[(size_t)q] = (int32_t)(rank_of(b1 ? e1 : e2) << 2) | (b1 ? 1 : 0) | (b2 ? 2 : 0);
      }
    }
  }
  return PYJAC_OK;
}

}  // namespace pyjac
