// Internal definitions shared by the host preprocessing (pyjac_host.cpp), the kernels
// (pyjac_kernels.cu) and the C ABI (pyjac_capi.cu).  Not part of the public boundary.
#pragma once
#include <cstdint>
#include <string>
#include <vector>

#include "pyjac.h"

namespace pyjac {

constexpr double R_GAS = 8314.46261815324;  // J/(kmol K)   DESIGN.md R1
constexpr double P_ATM = 101325.0;          // Pa

// bit fields of RxTables::info
constexpr int INFO_TYPE_MASK = 7;    // bits 0-2  reaction type
constexpr int INFO_REV = 1 << 3;     // reversible
constexpr int INFO_T2 = 1 << 4;      // Troe has T2
constexpr int INFO_ADEF = 1 << 5;    // default third-body efficiency is 1 (mixture); 0: single collider
constexpr int INFO_SIMPLE = 1 << 6;  // every stoichiometric coefficient is 1 (fast path, no powers)
constexpr int INFO_CHEM = 1 << 7;    // chemically-activated falloff: Arrhenius columns hold k_0, the falloff record k_inf
constexpr int INFO_REVX = 1 << 24;   // explicit reverse Arrhenius parameters (rev_par)
constexpr int INFO_FAST = 1 << 25;   // fast path of the reaction phase: elementary or third body, every coefficient 1, at most two
                                     // species per side, K_c-based reverse rate, the last species in no role
constexpr int INFO_SNU_SHIFT = 8;    // bits 8-11: sum(nu) + 8
constexpr int INFO_NREAC_SHIFT = 12; // bits 12-13: number of reactant entries
constexpr int INFO_NPROD_SHIFT = 14; // bits 14-15: number of product entries
constexpr int INFO_OF_SHIFT = 16;    // bits 16-19: forward order  sum nu'
constexpr int INFO_OR_SHIFT = 20;    // bits 20-23: reverse order  sum nu''
constexpr uint32_t SIGN_BIT = 0x80000000u;
constexpr int N_ZERO_SLOTS = 16;             // always-zero slots after the real ones: ELL padding, one per 8-byte bank
constexpr int XPAIR_PAD = 32 * 16;      // dense by expansion: pairs per batch (32 lanes x XIT warp iterations)
constexpr int SEG_LEN = 24;           // gather lists longer than this are split into segments

enum OutFmt { OUT_CSR = 0, OUT_CSC = 1, OUT_DENSE_C = 2, OUT_DENSE_F = 3 };

constexpr int ELL_W = 128;           // items per ELL super-group (4 items per lane at one state per CTA)
constexpr int ELL_W_NARROW = 512;   // items per NARROW super-group (segments of <= NARROW_LEN entries; species rows only)
constexpr int NARROW_LEN = 2;

struct GatherPlan {
  int stride = 1;                            // ints per entry
  bool packed = false, packable = true;      // stride 1: two 16-bit entries per word (see build_gather)
  int n_sg = 0;                              // ELL super-groups: n_wide of ELL_W segments, then n_sg - n_wide of ELL_W_NARROW
  int n_wide = 0;
  std::vector<int32_t> sg_meta;              // [n_sg*2]: entry offset, padded segment length (in words if packed)
  std::vector<int32_t> ell_ent;              // entry (p, w) of group sg at (off + p*ELL_W + w) * stride; packed: word (q, w) at off + q*ELL_W + w
  // processing slot (n_sg*ELL_W) -> what the segment's sum is: item id >= 0 (the whole list of that item: store
  // the result), -1 padding, <= -2: partial sum number -2 - target of a list that was split into segments
  std::vector<int32_t> target;
  int n_part = 0;                            // partial sums (shared-memory scratch)
  std::vector<int32_t> comb_item, comb_first, comb_nseg;   // split lists: item id, first partial, number of partials
  int64_t n_entries = 0, n_padded = 0;       // real / stored entries (padding overhead report)
};

// ---- host-side tables (reactions in SORTED order: by type, then reversibility) ------------------
struct HostTables {
  int ns = 0, nr = 0, nvar = 0;
  std::vector<int32_t> perm;                 // sorted index -> original reaction index
  // reaction chunks of phase 1 for S = 1, 2, 4, .. 32 states per CTA (index log2 S): chunk c = sorted reactions
  // [rxc[2c], rxc[2c+1]), at most 32 / S of them, never two cost groups (reaction type / fast path) in one chunk: a warp
  // that mixes two types runs both code paths one after the other, and the longest chunk bounds the phase
  std::vector<int32_t> rxc[6];
  // species
  std::vector<double> nasa;                  // [15*ns] coefficient-major: tmid, lo[7], hi[7]
  std::vector<double> wr;                    // [ns] W_k / W_Ns
  // reactions
  std::vector<double> lnA, beta, Ta, dn;     // [nr]; dn = sum_k<Ns nu_ki (1 - W_k/W_Ns)
  std::vector<int32_t> info, aux;            // [nr]; aux = index into fall / plog / cheb tables
  std::vector<uint32_t> sp;                  // [nr*8]: 0-2 reactants, 3-5 products: species | nu << 16; unused: species = ns (dummy), nu = 0
  std::vector<int32_t> eff_ptr, eff_sp;      // [nr+1], entries with alpha != default only
  std::vector<double> eff_d;                 // alpha - default
  std::vector<int32_t> slot_base;            // [nr+1] Jacobian slots: {T, E, reactant roles, product roles (rev), eff roles}
  std::vector<double> rev_par;               // [nr*3] ln A_r, beta_r, Ta_r of reactions with INFO_REVX (else 0); empty if none
  std::vector<double> fall;                  // [nf*12]: lnA0, beta0, Ta0, pad, then 5 blend parameters
  std::vector<int32_t> plog_ptr;             // [npl+1] pressure LEVELS of every P-Log reaction
  std::vector<int32_t> plog_ent;             // [n_levels+1] entries of every level (equal-pressure entries: rates summed, R10)
  std::vector<double> plog_P, plog_lnP;      // [n_levels]
  std::vector<double> plog_lnA, plog_b, plog_Ta;   // [n_entries]
  std::vector<int32_t> cheb_meta;            // [nc*4]: nT, nP, coef offset, 0
  std::vector<double> cheb_lim, cheb_coef;   // [nc*4]: 1/Tmin, 1/Tmax, log10 Pmin, log10 Pmax
  // pattern
  int64_t nnz = 0;
  std::vector<int32_t> csr_ptr, csr_idx, csc_ptr, csc_idx;
  std::vector<int32_t> csc2csr;              // [nnz] CSR value position of CSC entry p (finite-difference kernel)
  // gather plans.  Entries: slot offset | SIGN_BIT (a stoichiometric coefficient of magnitude m is m copies)
  int nA = 0;                                // number of species-block nonzeros
  GatherPlan jplan;                          // species rows: block nonzeros + their T and E columns
  GatherPlan cplan;                          // T and E rows, species columns: pairs (slot | sign, reaction)
  GatherPlan qplan;                          // source terms: omega_k gathers q_i
  std::vector<int32_t> j_pos[4];             // [OutFmt][jplan slots] output element; -1 padding; <= -2: partial -2 - x
  std::vector<int32_t> c_pos[4];             // [OutFmt][2 * cplan slots]: (T, j), (E, j); same encoding in [2*slot]
  std::vector<int32_t> jc_pos[4], cc_pos[4]; // [OutFmt] output elements of the split (combined) lists: [n_comb], [2*n_comb]
  std::vector<int32_t> q_target;             // qplan: slot -> species (>= 0), -1, or partial code
  int n_part_jac = 0, n_part_src = 0;        // doubles of partial-sum scratch per state
  int32_t d_pos[4][4];                       // (T,T) (T,E) (E,T) (E,E)
  std::vector<uint32_t> nzmask[2];           // dense bitmaps, bit e set iff dense element e ('C' / 'F' order) is in the pattern
  // dense by expansion: per 16-byte-aligned pair of dense elements (pair p = elements 2p - sh, 2p - sh + 1; sh = 0 / 1:
  // the matrix starts on an even / odd double) rank << 2 | present bits -- rank = CSR ('C') / CSC ('F') position of the
  // pair's first present element.  Index [2 * layout + sh]; padded with zeros to a multiple of XPAIR_PAD entries.
  std::vector<int32_t> xpair[4];
  int nslots = 0;                            // total Jacobian slots
  int max_eff = 0;
  // raw gather lists in the slot numbering above, consumed by build_jac_tables (pyjac_plan.cpp)
  std::vector<std::vector<int32_t>> raw_blk;  // [nA] species-block nonzero -> entries (slot | sign), |nu| copies
  std::vector<int32_t> blk_r, blk_c;          // [nA] matrix row / column of the nonzero
  std::vector<std::vector<int32_t>> raw_col;  // [Ns-1] species k -> entries (slot_base[r] | sign): T and E columns
  std::vector<std::vector<int32_t>> raw_row;  // [Ns-1] species j -> pairs (slot | sign, reaction): T and E rows
  std::vector<int32_t> csr2csc;               // [nnz] CSC value position of CSR entry p
};

// returns PYJAC_OK or an error code with a message in err
// approx: the "approximate" Jacobian of PAPER.md L313-317 (derivatives through the last species' concentration with
// respect to the other species' moles are ignored: sparser pattern, inexact values)
int build_host_tables(const pyjac_mech_desc* d, bool approx, HostTables& h, std::string& err);

// ---- analytical Jacobian kernel (pyjac_jacobian.cuh): block-partitioned plan -----------------------------------
// A thread owns one item for a PAIR of states (double2 everywhere).  The reactions are cut into H blocks so that the
// per-reaction partials ("slots") of one block and two states fit in shared memory; a gather list is cut into PIECES,
// one per (block, segment of <= J_SEG entries).  Pieces of one block are packed in groups of J_GW (ELL, padded,
// entry-pair-major); a group is homogeneous in kind and class and stores its plus entries before its minus entries.
constexpr int J_GW = 128;             // pieces per group
constexpr int J_GW1 = 256;            // pieces per group of kind JK_BLK1 (lists of exactly one entry)
constexpr int J_SEG = 24;             // longest piece (entries)
constexpr int J_NZERO = 16;           // always-zero value slots: ELL padding points at the first 8 (one per 16-byte bank group); the JK_COL gather also reads slot + 8
constexpr uint32_t J_NOPOS = 0xffffffffu;
// kind of a piece: species-block nonzero; the same with exactly one entry; T and E columns of a species row (two
// sums, slots v and v + 8); T and E rows of a species column (two sums weighted by dE~_i, dn~_i of the entry's
// reaction); JK_ROWC: combine of T/E-row partial sums (gathers like JK_COL, finishes like JK_ROW)
enum JKind { JK_BLK = 0, JK_BLK1 = 1, JK_COL = 2, JK_ROW = 3, JK_ROWC = 4 };
// class of a piece: store the finished value; partial = sum; partial += sum; store partial + sum
enum JCls { JC_OUT = 0, JC_FIRST = 1, JC_ADD = 2, JC_LAST = 3 };
// nP2 / nM2: pair steps of plus / minus entries (JK_ROW; JK_BLK1: 1 / 0 or 0 / 1); JK_BLK, JK_COL, JK_ROWC: nP2 = pair
// steps of the longest piece, nM2 = 0, and every piece has its own boundary (JacTables::nplus)
// qsteps: byte q = pair steps (of plus entries for JK_ROW) needed by pieces 32 q .. 32 q + 31
struct JGroup { uint32_t ent_off, piece_off; uint8_t nP2, nM2, cls, kind; uint32_t qsteps; };   // 16 bytes
// bits of JacTables::info
constexpr uint32_t JI_TYPE_MASK = 7, JI_REV = 1u << 3, JI_T2 = 1u << 4, JI_ADEF = 1u << 5, JI_FAST = 1u << 6, JI_CHEM = 1u << 7;
constexpr int JI_SNU_SHIFT = 8;       // bits 8-12: sum(nu) + 16
constexpr int JI_NREAC_SHIFT = 13, JI_NPROD_SHIFT = 15, JI_OF_SHIFT = 17, JI_OR_SHIFT = 21;
constexpr uint32_t JI_REVX = 1u << 25, JI_HASL = 1u << 26;

struct JacTables {
  int ns = 0, nr = 0, nvar = 0, H = 1;
  std::vector<int32_t> old_of_new;           // new reaction index -> index in the HostTables order
  std::vector<int32_t> blk_r0;               // [H+1] first reaction of every block
  std::vector<int32_t> blk_ng;               // [H] reactions of the block that take the general path of phase 1 (they come first)
  std::vector<double> lnA, beta, Ta, dn;     // [nr]
  std::vector<uint32_t> info;                // [nr]
  std::vector<uint32_t> sp;                  // [nr*4]: species 0|1, 2|3, 4|5 (16 bits each; unused = ns), slot base | nu bits << 16
  std::vector<int32_t> ext;                  // [nr*4]: aux, first efficiency, number of efficiencies, HostTables index
  int ns_max = 0;                            // value slots of the largest block (multiple of 8)
  int n_part = 0;                            // partial-sum slots
  int n_val = 0;                             // value space: ns_max + J_NZERO + n_part   (<= 65535: 16-bit entries)
  int max_nrb = 0;                           // reactions of the largest block
  std::vector<JGroup> groups;                // block by block, descending cost inside a block
  std::vector<int32_t> blk_g0;               // [H+2]; block H = the final combine wave
  std::vector<uint32_t> ent;                 // entries
  std::vector<uint32_t> posA[4], posB[4];    // [OutFmt][piece slot] output element (J_NOPOS: none)
  std::vector<uint16_t> pidx, item;          // [piece slot] partial slot; species column (JK_ROW, JK_ROWC)
  std::vector<uint8_t> nplus;                // [piece slot] JK_BLK / JK_COL / JK_ROWC: pair steps of plus entries (then minus)
  int n_pieces = 0;
  int32_t d_pos[4][4];
  int64_t n_entries = 0, n_padded = 0;       // real / stored entries
  int n_span = 0;                            // lists with more than one piece
};
constexpr int J_NT = 512, J_NW = J_NT / 32;   // threads / warps of the Jacobian kernel
constexpr int J_NSC = 24;                     // per-pair scalars kept in shared memory
constexpr int J_NRED = 12;                    // reduction words per warp: 0-6 reaction sums, 8-10 species sums
constexpr int J_MAXH = 8;
// bytes of dynamic shared memory of the Jacobian kernel with LS state pairs per item
size_t jac_smem_bytes(const JacTables& j, int LS);
constexpr size_t J_SMEM_LIMIT = 227 * 1024 - 256;   // dynamic part; the rest: static counters
// builds the plan with the smallest H whose footprint at one state pair per item fits; PYJAC_ENOMEM if none does
int build_jac_tables(const HostTables& h, JacTables& j, std::string& err);

// ---- device views ------------------------------------------------------------------------------
struct DevGather {
  int n_sg, n_wide, n_comb, part_base;   // part_base: offset of this plan's partial sums in the scratch
  const int32_t *sg_meta, *ell_ent, *comb_first, *comb_nseg;
};

struct DevMech {
  int ns, nr, nvar, nslots, n_part_jac, n_part_src;
  const double *nasa, *wr;
  const double *lnA, *beta, *Ta, *dn;
  const int32_t *info, *aux;
  const uint32_t* sp;
  const int32_t *eff_ptr, *eff_sp;
  const double* eff_d;
  const int32_t* slot_base;
  const int32_t* rxc[6];     // reaction chunks (first, end) of phase 1 per log2 S, n_rxc[] of them
  int n_rxc[6];
  const double* rev_par;
  const double* fall;
  const int32_t *plog_ptr, *plog_ent;
  const double *plog_P, *plog_lnP, *plog_lnA, *plog_b, *plog_Ta;
  const int32_t* cheb_meta;
  const double *cheb_lim, *cheb_coef;
  DevGather cplan, qplan;
  const int32_t *q_target, *c_item, *qc_item, *cc_item;   // slot -> species / column; combined lists -> species / column
  const int32_t *csc_ptr, *csc_idx, *csc2csr;             // pattern by columns (finite-difference kernel)
};

struct DevPlan {
  int64_t n_e;               // elements per state in the output (nnz or nvar^2)
  DevGather jplan;
  const int32_t *j_pos, *c_pos, *jc_pos, *cc_pos;
  int32_t d_pos[4];
  const uint32_t* nzmask;    // dense only (else nullptr)
  // dense by expansion (jacobian_kernel MODE 2, else nullptr): pair tables and n_sm x 2 x nnz doubles of scratch
  const int32_t* xpair[2];   // dense by expansion: the pair tables of this layout for sh = 0 / 1 (HostTables::xpair)
  double* scratch;
};

// device view of JacTables (+ the type-specific parameter tables it shares with DevMech)
struct DevJac {
  int ns, nr, nvar, H, ns_max, n_val, max_nrb, n_groups;
  int blk_r0[J_MAXH + 1], blk_ng[J_MAXH], blk_g0[J_MAXH + 2];
  const double *lnA, *beta, *Ta, *dn;
  const uint32_t* info;
  const uint32_t* sp;         // uint4 per reaction
  const int32_t* ext;         // int4 per reaction
  const JGroup* groups;
  const uint32_t* ent;
  const uint16_t *pidx, *item;
  const uint8_t* nplus;
  const double* nasa;
  const int32_t* eff_sp;
  const double* eff_d;
  const double* rev_par;
  const double* fall;
  const int32_t *plog_ptr, *plog_ent;
  const double *plog_P, *plog_lnP, *plog_lnA, *plog_b, *plog_Ta;
  const int32_t* cheb_meta;
  const double *cheb_lim, *cheb_coef;
};
struct DevJacOut {
  int64_t n_e;                // elements per state in the output (nnz or nvar^2)
  const void *posA, *posB;    // uint16_t (pos16) or uint32_t per piece slot
  int pos16;
  int32_t d_pos[4];
  const uint32_t* nzmask;     // dense only (else nullptr)
};

struct LaunchCfg { int S, threads; size_t smem; };

// what: 0 source, 1 jacobian.  Chooses states-per-CTA from the shared-memory footprint and `tile`.
constexpr size_t SMEM_LIMIT = 227 * 1024 - 64;   // dynamic shared memory of the tile kernels; 64 B left for static counters
// n_sm: SMs of the handle's device (states per CTA are reduced until there are two tiles per SM)
LaunchCfg choose_cfg(const HostTables& h, bool jac, int64_t tile, int64_t n_states, int n_sm);

// kernel launchers (pyjac_kernels.cu); return cudaError_t as int
int launch_source(const DevMech& m, const LaunchCfg& cfg, int mode, int64_t n_states, int64_t ld, int64_t tile,
                  const double* phi, const double* param, double* out, void* stream);
int launch_jacobian(const DevMech& m, const DevPlan& p, const LaunchCfg& cfg, int mode, int64_t n_states, int64_t ld,
                    int64_t tile, const double* phi, const double* param, double* out, unsigned long long* sched, void* stream);
// the pair-of-states Jacobian kernel (pyjac_jacobian.cuh).  LS = state pairs per item (1, 2 or 4: 2 LS states per CTA)
LaunchCfg choose_cfg_jac(const JacTables& j, int64_t tile, int64_t n_states, int n_sm);
int launch_jacobian2(const DevJac& m, const DevJacOut& o, const LaunchCfg& cfg, int n_sm, int mode, int64_t n_states, int64_t tile,
                     const double* phi, const double* param, double* out, unsigned long long* sched, void* stream);
int set_kernel_attributes_jac();
// sched: two zero-initialised 64-bit words in device memory (tile counter, finished CTAs) that no other launch in
// flight uses; the kernel leaves them zero again.
// first-order forward finite-difference Jacobian.  ofmt: OutFmt.  S = columns per pass.
LaunchCfg choose_cfg_fd(const HostTables& h);
int launch_fd(const DevMech& m, const LaunchCfg& cfg, int mode, int ofmt, int64_t n_e, double rel_step, double abs_step,
              int64_t n_states, int64_t ld, int64_t tile, const double* phi, const double* param, double* out, void* stream);
int set_kernel_attributes();

}  // namespace pyjac
