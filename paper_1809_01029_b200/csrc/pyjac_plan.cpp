// Step a0, second part (one-time, host): the block-partitioned gather plan of the analytical Jacobian kernel
// (pyjac_jacobian.cuh).  Input: the tables, pattern and raw gather lists of build_host_tables (pyjac_host.cpp).
//
// J = W G (R4-8): every nonzero is a static list of per-reaction partials ("slots") with signs.  This is
// the static full-index -> sparse-index map the paper proposes instead of its run-time CRS/CCS search (PAPER.md
// L345, L559).  New here: the reactions are cut into H blocks so that the slots of ONE block for TWO states fit in
// shared memory next to everything else; lists that span blocks carry a partial sum from block to block.
#include <algorithm>
#include <array>
#include <cstring>
#include <functional>
#include <map>
#include <numeric>
#include <sstream>

#include "pyjac_internal.h"

namespace pyjac {

namespace {

struct Piece {
  int kind, cls, block;
  std::vector<uint32_t> P, M;       // entries: value slot (| reaction-in-block << 16 for JK_ROW)
  int pidx = 0;                     // partial slot (classes FIRST / ADD / LAST)
  int r = -1, c = -1, c2 = -1, r2 = -1;   // output coordinates: (r, c) -> posA, (r2, c2) -> posB
  int item = 0;
};

int len2(size_t n) { return (int)((n + 1) / 2); }

}  // namespace

size_t jac_smem_bytes(const JacTables& j, int LS) {
  const size_t pair16 = 2 * (size_t)J_NSC + 4 * (size_t)(j.ns + 1) + (size_t)j.max_nrb + (size_t)j.n_val + (size_t)J_NW * J_NRED;
  return 16 * (size_t)LS * pair16 + 8 * (size_t)((j.nr + 1) & ~1) + 16 * j.groups.size();
}

static int build_with_blocks(const HostTables& h, int H, JacTables& j, std::string& err) {
  const int ns = h.ns, nr = h.nr, L = ns - 1;
  j = JacTables();
  j.ns = ns; j.nr = nr; j.nvar = h.nvar; j.H = H;
  auto nslots_of = [&](int r_old) { return h.slot_base[r_old + 1] - h.slot_base[r_old]; };
  auto species_of = [&](int r_old, int a) { return (int)(h.sp[8 * r_old + a] & 0xffff); };

  // ---- 1. partition: reactions ordered by their RAREST species (reactions that share an unpopular species end up in
  // the same block, which keeps most short lists inside one block), cut into H runs of equal slot count -------------
  std::vector<int> pop(ns + 1, 0);
  for (int r = 0; r < nr; ++r) for (int a = 0; a < 6; ++a) pop[species_of(r, a)]++;
  std::vector<int> order(nr);
  std::iota(order.begin(), order.end(), 0);
  std::vector<int> blk_of_old(nr, 0);
  if (H > 1) {
    std::vector<int> key(nr, 0);
    for (int r = 0; r < nr; ++r) {
      int best = -1;
      for (int a = 0; a < 6; ++a) {
        const int k = species_of(r, a);
        if (k >= L) continue;               // dummy entry or the last species
        if (best < 0 || pop[k] < pop[best] || (pop[k] == pop[best] && k < best)) best = k;
      }
      key[r] = best < 0 ? ns : best;
    }
    std::stable_sort(order.begin(), order.end(), [&](int a, int b) { return key[a] < key[b]; });
    int64_t total = 0, run = 0;
    for (int r = 0; r < nr; ++r) total += nslots_of(r);
    for (int q = 0; q < nr; ++q) {
      blk_of_old[order[q]] = (int)std::min<int64_t>(H - 1, run * H / total);
      run += nslots_of(order[q]);
    }
  }
  // inside a block: the reactions of the general path of phase 1 first (the kernel gives them a lane per STATE and
  // hands them out first: they are the expensive ones), then the fast-path reactions; inside each part the HostTables
  // order (descending cost class, bank-friendly inside a class) is kept
  auto is_fast = [&](int ro) {
    const int oi = h.info[ro];
    const int type = oi & INFO_TYPE_MASK, nre = (oi >> INFO_NREAC_SHIFT) & 3, npr = (oi >> INFO_NPROD_SHIFT) & 3;
    bool hasL = false;
    for (int a = 0; a < 6; ++a) hasL |= species_of(ro, a) == L;
    for (int e = h.eff_ptr[ro]; e < h.eff_ptr[ro + 1]; ++e) hasL |= h.eff_sp[e] == L;
    return (type == PYJAC_ELEMENTARY || type == PYJAC_THIRD_BODY) && (oi & INFO_SIMPLE) && nre <= 2 && npr <= 2 && !(oi & INFO_REVX) && !hasL;
  };
  std::vector<std::vector<int>> members(H);
  for (int pass = 0; pass < 2; ++pass)
    for (int r = 0; r < nr; ++r)
      if ((int)is_fast(r) == pass) members[blk_of_old[r]].push_back(r);
  j.blk_r0.assign(1, 0);
  std::vector<int> new_of_old(nr, 0);
  for (int b = 0; b < H; ++b) {
    int ng = 0;
    for (int r : members[b]) { new_of_old[r] = (int)j.old_of_new.size(); j.old_of_new.push_back(r); ng += is_fast(r) ? 0 : 1; }
    j.blk_r0.push_back((int)j.old_of_new.size());
    j.blk_ng.push_back(ng);
    j.max_nrb = std::max(j.max_nrb, (int)members[b].size());
  }
  for (int b = 0; b < H; ++b)
    if (members[b].empty()) { err = "internal: empty reaction block"; return PYJAC_EMECH; }

  // ---- 2. value slots: reactions in groups of 8, slot i of reaction lr at base + 8 i + lr % 8 (the 8 lanes of a
  // quarter-warp store 8 consecutive 16-byte words: no bank conflicts in phase 1) ------------------------------------
  std::vector<int> sb(nr, 0);      // slot base of the new reaction index (relative to its block)
  for (int b = 0; b < H; ++b) {
    int base = 0;
    const int r0 = j.blk_r0[b], r1 = j.blk_r0[b + 1];
    for (int g0 = r0; g0 < r1; g0 += 8) {
      int w = 0;
      for (int r = g0; r < std::min(g0 + 8, r1); ++r) w = std::max(w, nslots_of(j.old_of_new[r]));
      for (int r = g0; r < std::min(g0 + 8, r1); ++r) sb[r] = base + (r - g0);
      base += 8 * w;
    }
    j.ns_max = std::max(j.ns_max, base);
  }
  if (j.ns_max + J_NZERO > 65535) { err = "mechanism too large: value slots of a block exceed 16 bits"; return PYJAC_ENOMEM; }
  std::vector<int> owner(h.nslots, 0);
  for (int r = 0; r < nr; ++r) for (int s = h.slot_base[r]; s < h.slot_base[r + 1]; ++s) owner[s] = r;
  struct Ref { int block; uint32_t v; bool minus; };
  auto translate = [&](int32_t e) {
    const uint32_t u = (uint32_t)e;
    const int s = (int)(u & ~SIGN_BIT), r_old = owner[s], rn = new_of_old[r_old];
    return Ref{blk_of_old[r_old], (uint32_t)(sb[rn] + 8 * (s - h.slot_base[r_old])), (u & SIGN_BIT) != 0};
  };

  // ---- 3. reaction tables in the new order ------------------------------------------------------------------------
  j.lnA.resize(nr); j.beta.resize(nr); j.Ta.resize(nr); j.dn.resize(nr); j.info.resize(nr);
  j.sp.resize((size_t)nr * 4); j.ext.resize((size_t)nr * 4);
  for (int rn = 0; rn < nr; ++rn) {
    const int ro = j.old_of_new[rn];
    j.lnA[rn] = h.lnA[ro]; j.beta[rn] = h.beta[ro]; j.Ta[rn] = h.Ta[ro]; j.dn[rn] = h.dn[ro];
    const int oi = h.info[ro];
    const int nre = (oi >> INFO_NREAC_SHIFT) & 3, npr = (oi >> INFO_NPROD_SHIFT) & 3;
    const int snu = ((oi >> INFO_SNU_SHIFT) & 15) - 8;
    const int of = (oi >> INFO_OF_SHIFT) & 15, orv = (oi >> INFO_OR_SHIFT) & 15;
    const int type = oi & INFO_TYPE_MASK;
    uint32_t nu_bits = 0;
    bool hasL = false;
    for (int a = 0; a < 6; ++a) {
      nu_bits |= ((h.sp[8 * ro + a] >> 16) & 3u) << (2 * a);
      hasL |= species_of(ro, a) == L;
    }
    for (int e = h.eff_ptr[ro]; e < h.eff_ptr[ro + 1]; ++e) hasL |= h.eff_sp[e] == L;
    // fast path of phase 1: elementary or third body, every coefficient 1, at most two species per side, K_c-based
    // reverse rate, the last species not involved in any role
    const bool fast = is_fast(ro);
    uint32_t info = (uint32_t)type | ((oi & INFO_REV) ? JI_REV : 0u) | ((oi & INFO_T2) ? JI_T2 : 0u) | ((oi & INFO_ADEF) ? JI_ADEF : 0u) |
                    ((oi & INFO_CHEM) ? JI_CHEM : 0u) | (fast ? JI_FAST : 0u) | ((uint32_t)(snu + 16) << JI_SNU_SHIFT) |
                    ((uint32_t)nre << JI_NREAC_SHIFT) | ((uint32_t)npr << JI_NPROD_SHIFT) | ((uint32_t)of << JI_OF_SHIFT) |
                    ((uint32_t)orv << JI_OR_SHIFT) | ((oi & INFO_REVX) ? JI_REVX : 0u) | (hasL ? JI_HASL : 0u);
    j.info[rn] = info;
    for (int w = 0; w < 3; ++w)
      j.sp[4 * rn + w] = (uint32_t)species_of(ro, 2 * w) | ((uint32_t)species_of(ro, 2 * w + 1) << 16);
    j.sp[4 * rn + 3] = (uint32_t)sb[rn] | (nu_bits << 16);
    j.ext[4 * rn] = h.aux[ro]; j.ext[4 * rn + 1] = h.eff_ptr[ro]; j.ext[4 * rn + 2] = h.eff_ptr[ro + 1] - h.eff_ptr[ro];
    j.ext[4 * rn + 3] = ro;
  }

  // ---- 4. pieces --------------------------------------------------------------------------------------------------
  std::vector<Piece> pieces;
  int n_part1 = 0, n_part2 = 0;       // single-valued / two-valued partial chains
  // partial slot numbers are assigned after counting: single chains first, then the two-valued ones in groups of 8
  // chains (value 0 at base + c % 8, value 1 at + 8: the layout the JK_COL gather reads)
  struct Chain { bool two; int idx; };
  std::vector<Chain> chains;
  auto new_chain = [&](bool two) { chains.push_back({two, two ? n_part2++ : n_part1++}); return (int)chains.size() - 1; };
  // entries per block of one list -> pieces.  kind: JK_BLK / JK_COL / JK_ROW; must_end_last: the list may only be
  // finished in the last block (T and E rows need f_T, known when every reaction is done).
  auto add_list = [&](int kind, const std::vector<std::vector<std::pair<uint32_t, bool>>>& per_block, int r, int c, int r2, int c2, int item) {
    const bool two = kind != JK_BLK;
    const bool must_end_last = kind == JK_ROW;
    struct Seg { int block; std::vector<uint32_t> P, M; };
    std::vector<std::vector<Seg>> segs(H);
    int n_pieces_total = 0, w = 0, last_block = -1;
    for (int b = 0; b < H; ++b) {
      const auto& v = per_block[b];
      if (v.empty()) continue;
      last_block = b;
      // plus entries first, then minus; cut the concatenation into nearly equal segments of <= J_SEG entries
      std::vector<std::pair<uint32_t, bool>> seq;
      for (auto& e : v) if (!e.second) seq.push_back(e);
      for (auto& e : v) if (e.second) seq.push_back(e);
      const int len = (int)seq.size(), nseg = (len + J_SEG - 1) / J_SEG;
      for (int q = 0; q < nseg; ++q) {
        Seg s; s.block = b;
        const int a0 = (int)((int64_t)len * q / nseg), a1 = (int)((int64_t)len * (q + 1) / nseg);
        for (int t = a0; t < a1; ++t) (seq[t].second ? s.M : s.P).push_back(seq[t].first);
        segs[b].push_back(std::move(s));
      }
      n_pieces_total += nseg; w = std::max(w, nseg);
    }
    if (must_end_last && last_block != H - 1) { segs[H - 1].push_back(Seg{H - 1, {}, {}}); ++n_pieces_total; w = std::max(w, 1); last_block = H - 1; }
    if (n_pieces_total == 0) {           // an empty list still has an output (e.g. an inert species' T column entry)
      segs[H - 1].push_back(Seg{H - 1, {}, {}}); n_pieces_total = 1; w = 1; last_block = H - 1;
    }
    auto make = [&](Seg& s, int cls, int pidx_chain) {
      Piece p; p.kind = kind; p.cls = cls; p.block = s.block; p.P = std::move(s.P); p.M = std::move(s.M);
      p.pidx = pidx_chain; p.r = r; p.c = c; p.r2 = r2; p.c2 = c2; p.item = item;
      if (kind == JK_BLK && cls == JC_OUT && p.P.size() + p.M.size() == 1) p.kind = JK_BLK1;
      pieces.push_back(std::move(p));
    };
    if (n_pieces_total == 1) { make(segs[last_block][0], JC_OUT, -1); return; }
    j.n_span++;
    if (w == 1) {                        // one chain: first ... add ... last
      const int ch = new_chain(two);
      bool first = true;
      for (int b = 0; b < H; ++b)
        for (Seg& s : segs[b]) { make(s, b == last_block ? JC_LAST : (first ? JC_FIRST : JC_ADD), ch); first = false; }
      return;
    }
    // several segments in some block: chain q takes segment q of every block; a combine piece in the final wave
    std::vector<int> ch(w, -1);
    Seg comb; comb.block = H;
    for (int b = 0; b < H; ++b)
      for (size_t q = 0; q < segs[b].size(); ++q) {
        const bool first = ch[q] < 0;
        if (first) ch[q] = new_chain(two);
        make(segs[b][q], first ? JC_FIRST : JC_ADD, ch[q]);
      }
    Piece p; p.kind = kind == JK_ROW ? JK_ROWC : kind; p.cls = JC_OUT; p.block = H; p.pidx = -1;
    p.r = r; p.c = c; p.r2 = r2; p.c2 = c2; p.item = item;
    for (int q = 0; q < w; ++q) p.P.push_back(0x80000000u | (uint32_t)ch[q]);     // chain reference, resolved below
    pieces.push_back(std::move(p));
  };
  {
    std::vector<std::vector<std::pair<uint32_t, bool>>> pb(H);
    for (int i = 0; i < h.nA; ++i) {
      for (auto& v : pb) v.clear();
      for (int32_t e : h.raw_blk[i]) { const Ref f = translate(e); pb[f.block].push_back({f.v, f.minus}); }
      add_list(JK_BLK, pb, h.blk_r[i], h.blk_c[i], -1, -1, 0);
    }
    for (int k = 0; k < L; ++k) {
      for (auto& v : pb) v.clear();
      for (int32_t e : h.raw_col[k]) { const Ref f = translate(e); pb[f.block].push_back({f.v, f.minus}); }
      add_list(JK_COL, pb, 2 + k, 0, 2 + k, 1, k);
    }
    for (int jc = 0; jc < L; ++jc) {
      for (auto& v : pb) v.clear();
      for (size_t e = 0; e + 1 < h.raw_row[jc].size(); e += 2) {
        const Ref f = translate(h.raw_row[jc][e]);
        const int rn = new_of_old[h.raw_row[jc][e + 1]];
        pb[f.block].push_back({f.v | ((uint32_t)(rn - j.blk_r0[f.block]) << 16), f.minus});
      }
      add_list(JK_ROW, pb, 0, 2 + jc, 1, 2 + jc, jc);
    }
  }
  // partial slots: [single chains][trash single][two-valued chains in groups of 8 x 2][trash pair inside the last group]
  const int part0 = j.ns_max + J_NZERO;
  const int trash1 = part0 + n_part1;
  int base2 = trash1 + 1;
  base2 = (base2 + 7) & ~7;
  const int n2 = n_part2 + 1;                         // + trash pair
  auto slot_of_chain = [&](int ch) {
    const Chain& c = chains[ch];
    return c.two ? base2 + 16 * (c.idx / 8) + (c.idx % 8) : part0 + c.idx;
  };
  const int trash2 = base2 + 16 * (n_part2 / 8) + (n_part2 % 8);
  j.n_val = base2 + 16 * ((n2 + 7) / 8);
  j.n_part = j.n_val - part0;
  if (j.n_val > 65535) { err = "mechanism too large: value space exceeds 16 bits"; return PYJAC_ENOMEM; }
  for (Piece& p : pieces) {
    for (uint32_t& e : p.P) if (e & 0x80000000u) e = (uint32_t)slot_of_chain((int)(e & 0x7fffffffu));
    p.pidx = p.pidx >= 0 ? slot_of_chain(p.pidx) : 0;
  }

  // ---- 5. groups --------------------------------------------------------------------------------------------------
  auto csr_pos = [&](int r, int c) {
    auto b = h.csr_idx.begin() + h.csr_ptr[r], e = h.csr_idx.begin() + h.csr_ptr[r + 1];
    return (int)(std::lower_bound(b, e, c) - h.csr_idx.begin());
  };
  auto pos_of = [&](int fmt, int r, int c) -> uint32_t {
    if (r < 0) return J_NOPOS;
    switch (fmt) {
      case OUT_CSR: return (uint32_t)csr_pos(r, c);
      case OUT_CSC: return (uint32_t)h.csr2csc[csr_pos(r, c)];
      case OUT_DENSE_C: return (uint32_t)(r * h.nvar + c);
      default: return (uint32_t)(c * h.nvar + r);
    }
  };
  for (int f = 0; f < 4; ++f) {
    j.d_pos[f][0] = (int32_t)pos_of(f, 0, 0); j.d_pos[f][1] = (int32_t)pos_of(f, 0, 1);
    j.d_pos[f][2] = (int32_t)pos_of(f, 1, 0); j.d_pos[f][3] = (int32_t)pos_of(f, 1, 1);
  }
  j.blk_g0.assign(1, 0);
  std::vector<int> idx_all(pieces.size());
  std::iota(idx_all.begin(), idx_all.end(), 0);
  for (int b = 0; b <= H; ++b) {
    std::vector<int> mine;
    for (int i : idx_all) if (pieces[i].block == b) mine.push_back(i);
    auto klass = [&](const Piece& p) { return p.kind * 4 + p.cls; };
    std::stable_sort(mine.begin(), mine.end(), [&](int a, int c) {
      const Piece &x = pieces[a], &y = pieces[c];
      if (klass(x) != klass(y)) return klass(x) < klass(y);
      const int lx = len2(x.P.size()) + len2(x.M.size()), ly = len2(y.P.size()) + len2(y.M.size());
      if (lx != ly) return lx > ly;
      if (x.P.size() != y.P.size()) return x.P.size() > y.P.size();
      return false;
    });
    std::vector<JGroup> gb;
    struct Built { JGroup g; std::vector<uint32_t> ent; std::vector<int> members; std::vector<uint8_t> nplus; int cost = 0; };
    std::vector<Built> built;
    size_t i0 = 0;
    while (i0 < mine.size()) {
      const Piece& first = pieces[mine[i0]];
      const int GW = first.kind == JK_BLK1 ? J_GW1 : J_GW;
      size_t i1 = i0;
      while (i1 < mine.size() && (int)(i1 - i0) < GW && klass(pieces[mine[i1]]) == klass(first) &&
             (first.kind != JK_BLK1 || pieces[mine[i1]].P.size() == first.P.size())) ++i1;   // JK_BLK1: one sign per group
      Built B;
      B.members.assign(mine.begin() + i0, mine.begin() + i1);
      // JK_ROW (and JK_BLK1): one plus / minus boundary for the whole group (nP2 pair steps, then nM2).
      // JK_BLK / JK_COL / JK_ROWC: every piece has its own boundary (nplus pair steps of plus entries, the rest minus):
      // the group is padded to its longest piece only, whatever the split of each piece.
      const bool own_boundary = first.kind == JK_BLK || first.kind == JK_COL || first.kind == JK_ROWC;
      int nP2 = 0, nM2 = 0;
      for (int m : B.members) {
        const int p2 = len2(pieces[m].P.size()), m2 = len2(pieces[m].M.size());
        if (own_boundary) nP2 = std::max(nP2, p2 + m2);
        else { nP2 = std::max(nP2, p2); nM2 = std::max(nM2, m2); }
      }
      if (nP2 > 255 || nM2 > 255) { err = "internal: piece too long"; return PYJAC_EMECH; }
      B.g.nP2 = (uint8_t)nP2; B.g.nM2 = (uint8_t)nM2; B.g.cls = (uint8_t)first.cls; B.g.kind = (uint8_t)first.kind;
      // entry order inside a part is free: schedule every quarter-warp (8 pieces) step by step with a maximum bipartite
      // matching pieces <-> 16-byte bank groups (slot mod 8); padding takes a zero slot in a free bank group
      const int n_steps = 2 * (nP2 + nM2);
      std::vector<std::vector<uint32_t>> sched(GW, std::vector<uint32_t>(n_steps, 0));
      B.nplus.assign(GW, 0);
      for (int q0 = 0; q0 < GW; q0 += 8) {
        std::vector<uint32_t> remP[8], remM[8];
        int bnd[8];                                               // first minus step of the lane
        for (int l = 0; l < 8; ++l) {
          bnd[l] = 2 * nP2;
          if (q0 + l < (int)B.members.size()) {
            remP[l] = pieces[B.members[q0 + l]].P; remM[l] = pieces[B.members[q0 + l]].M;
            if (own_boundary) bnd[l] = 2 * len2(remP[l].size());
          } else if (own_boundary) bnd[l] = 0;
          B.nplus[q0 + l] = (uint8_t)(bnd[l] / 2);
        }
        for (int t = 0; t < n_steps; ++t) {
          std::vector<uint32_t>* rem[8];
          for (int l = 0; l < 8; ++l) rem[l] = t < bnd[l] ? &remP[l] : &remM[l];
          int own[8]; std::fill(own, own + 8, -1);                // bank group -> lane
          std::function<bool(int, uint32_t&)> augment = [&](int l, uint32_t& seen) -> bool {
            for (uint32_t e : *rem[l]) {
              const int bk = (int)(e & 7);
              if (seen >> bk & 1) continue;
              seen |= 1u << bk;
              if (own[bk] < 0 || augment(own[bk], seen)) { own[bk] = l; return true; }
            }
            return false;
          };
          std::vector<int> lanes;
          for (int l = 0; l < 8; ++l) if (!rem[l]->empty()) lanes.push_back(l);
          std::stable_sort(lanes.begin(), lanes.end(), [&](int a, int c) { return rem[a]->size() > rem[c]->size(); });
          for (int l : lanes) { uint32_t seen = 0; augment(l, seen); }
          int pick[8]; std::fill(pick, pick + 8, -1);
          uint32_t used = 0;
          for (int bk = 0; bk < 8; ++bk) if (own[bk] >= 0) pick[own[bk]] = bk;
          for (int l = 0; l < 8; ++l) {
            if (rem[l]->empty()) continue;
            size_t at = 0;
            if (pick[l] >= 0) for (size_t q = 0; q < rem[l]->size(); ++q) if ((int)((*rem[l])[q] & 7) == pick[l]) { at = q; break; }
            sched[q0 + l][t] = (*rem[l])[at];
            used |= 1u << ((*rem[l])[at] & 7);
            rem[l]->erase(rem[l]->begin() + at);
            j.n_entries++;
            pick[l] = -2;
          }
          for (int l = 0; l < 8; ++l) {
            if (pick[l] == -2) continue;
            int z = 0;
            for (int c = 0; c < 8; ++c) if (!(used >> c & 1)) { z = c; used |= 1u << c; break; }
            sched[q0 + l][t] = (uint32_t)(j.ns_max + z);          // JK_ROW: reaction 0 of the block, times zero
          }
        }
        for (int l = 0; l < 8; ++l)
          if (!remP[l].empty() || !remM[l].empty()) { err = "internal: gather schedule lost entries"; return PYJAC_EMECH; }
      }
      // storage: JK_BLK / JK_COL / JK_ROWC: word (step2, piece) = entry 2 step2 | entry 2 step2 + 1 << 16;
      // JK_ROW: two words per (step2, piece); JK_BLK1: 16-bit entries, piece-major
      if (first.kind == JK_BLK1) {
        B.ent.assign(GW / 2, 0);
        const bool minus = first.P.empty();
        B.g.nP2 = minus ? 0 : 1; B.g.nM2 = minus ? 1 : 0;
        for (int p = 0; p < GW; ++p) {
          uint32_t e = (uint32_t)j.ns_max + (uint32_t)(p & 7);
          if (p < (int)B.members.size()) e = minus ? pieces[B.members[p]].M[0] : pieces[B.members[p]].P[0];
          B.ent[p / 2] |= (e & 0xffffu) << (16 * (p & 1));
        }
        j.n_padded += GW;
      } else if (first.kind == JK_ROW) {
        B.ent.resize((size_t)n_steps * GW);
        for (int s2 = 0; s2 < n_steps / 2; ++s2)
          for (int p = 0; p < GW; ++p) {
            B.ent[((size_t)s2 * GW + p) * 2] = sched[p][2 * s2];
            B.ent[((size_t)s2 * GW + p) * 2 + 1] = sched[p][2 * s2 + 1];
          }
        j.n_padded += (int64_t)n_steps * GW;
      } else {
        B.ent.resize((size_t)(n_steps / 2) * GW);
        for (int s2 = 0; s2 < n_steps / 2; ++s2)
          for (int p = 0; p < GW; ++p) B.ent[(size_t)s2 * GW + p] = (sched[p][2 * s2] & 0xffffu) | (sched[p][2 * s2 + 1] << 16);
        j.n_padded += (int64_t)n_steps * GW;
      }
      // pair steps actually needed by every quarter of the group (32 pieces; the pieces are sorted by descending
      // length): the kernel stops a quarter's lanes there instead of running them to the group's longest piece
      B.g.qsteps = 0;
      int work = 0;
      for (int q = 0; q < 4; ++q) {
        int mx = 0;
        for (int p = 32 * q; p < std::min<int>(32 * q + 32, (int)B.members.size()); ++p) {
          const Piece& pc = pieces[B.members[p]];
          mx = std::max(mx, own_boundary ? len2(pc.P.size()) + len2(pc.M.size()) : len2(pc.P.size()));
        }
        B.g.qsteps |= (uint32_t)mx << (8 * q);
        work += mx + nM2;
      }
      j.n_padded -= first.kind == JK_BLK1 ? 0 : (int64_t)n_steps * GW - 64 * (int64_t)work;    // count what is gathered
      // descending cost: work per piece ~ entries x (loads per entry) + fixed epilogue
      const int wk = first.kind == JK_BLK || first.kind == JK_BLK1 ? 2 : (first.kind == JK_ROW ? 5 : 3);
      B.cost = first.kind == JK_BLK1 ? 40 : work * wk + 16;
      built.push_back(std::move(B));
      i0 = i1;
    }
    std::stable_sort(built.begin(), built.end(), [](const Built& a, const Built& c) { return a.cost > c.cost; });
    for (Built& B : built) {
      const int GW = B.g.kind == JK_BLK1 ? J_GW1 : J_GW;
      if (j.ent.size() & 1) j.ent.push_back(0);                   // 8-byte alignment (JK_ROW reads uint2)
      B.g.ent_off = (uint32_t)j.ent.size();
      B.g.piece_off = (uint32_t)j.n_pieces;
      j.ent.insert(j.ent.end(), B.ent.begin(), B.ent.end());
      for (int p = 0; p < GW; ++p) {
        const bool real = p < (int)B.members.size();
        const Piece* pc = real ? &pieces[B.members[p]] : nullptr;
        for (int f = 0; f < 4; ++f) {
          j.posA[f].push_back(real ? pos_of(f, pc->r, pc->c) : J_NOPOS);
          j.posB[f].push_back(real ? pos_of(f, pc->r2, pc->c2) : J_NOPOS);
        }
        const bool two = B.g.kind != JK_BLK && B.g.kind != JK_BLK1;
        j.pidx.push_back((uint16_t)(real ? pc->pidx : (two ? trash2 : trash1)));
        j.nplus.push_back(B.nplus[p]);
        j.item.push_back((uint16_t)(real ? pc->item : 0));
      }
      j.n_pieces += GW;
      j.groups.push_back(B.g);
    }
    j.blk_g0.push_back((int)j.groups.size());
  }
  return PYJAC_OK;
}

int build_jac_tables(const HostTables& h, JacTables& j, std::string& err) {
  for (int H = 1; H <= J_MAXH; ++H) {
    if (H > h.nr) break;
    const int rc = build_with_blocks(h, H, j, err);
    if (rc == PYJAC_OK && jac_smem_bytes(j, 1) <= J_SMEM_LIMIT) return PYJAC_OK;
    if (rc != PYJAC_OK && rc != PYJAC_ENOMEM) return rc;
  }
  err = "mechanism too large: the Jacobian kernel's per-state intermediates do not fit in shared memory";
  return PYJAC_ENOMEM;
}

}  // namespace pyjac
