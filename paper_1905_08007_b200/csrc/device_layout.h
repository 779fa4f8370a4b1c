// device_layout.h — plain-old-data layout of one prepared diagram as the kernels read it.
// Product code (libmcqed.so). Shares nothing with oracle/.
//
// One diagram = one contiguous blob of 8-byte words in HBM:
//   DevHeader | Z[2^M] | invDeg[2^M] | DevGeom[ngeom] | DevTable[ntable] | DevNode[nnode] | DevTerm[nterm] | streams
// A "stream" is the numerator table of one (piece, operator): a sequence of families.
#pragma once
#include <cstdint>

#define MQ_MAXL 5
#define MQ_MAXM 15
#define MQ_MAXSLOT 14
#define MQ_MAXCHILD 5
#define MQ_NGRADE 6
#define MQ_MAXGEOM 96
#define MQ_MAXNODE 96          // nodes of the term trees of one diagram (max over all 6354 five-loop graphs: 95)
#define MQ_MAXNODEVAL 544      // graded node values of one diagram (max over all five-loop graphs: 528)
#define MQ_MAXPAT 16      // 2^(max #S-children of a piece)
// inner dense binary dimensions of a family, by number of Wick pairs c (bounds the static code and the family size)
// kd <= 4 blocks are evaluated by one Horner pass in registers (8 partial values); kd = 5, 6 blocks are 2 / 4 such blocks
// combined over the top variables (two-stage Horner), so the register need does not grow. A larger kd merges the 2^(kd-4)
// families of a slot set that differ only in the P+/P- choice of outer lines: half the stream entries, a third fewer operand
// gathers and scalar factors at 5-loop for 3 % more stored coefficients (measured). Caps keep an entry of MQ_WL families
// below one chunk.
#ifndef MQ_KD4
#define MQ_KD4 2              // inner dimension cap of c = 4 families (1 lets an entry of 4 families fit a 1024-word chunk)
#endif
static inline int mq_kd_max(int c) { return c <= 2 ? 6 : c == 3 ? 4 : MQ_KD4; }
#define MQ_MAXSCAL 12
#ifndef MQ_WL
#define MQ_WL 4               // families per stream entry = lanes that share one point group (MQ_NP points in binary64, 1 in double-double)
#endif
#ifndef MQ_CHUNK_WORDS
#define MQ_CHUNK_WORDS (MQ_WL > 2 ? 2048 : 1024)   // staging granule of the family stream (8 / 16 KiB): the largest entry (MQ_WL families of c = 4, kd = 2) must fit
#endif
#define MQ_PAD_MARK 7        // header field c of a PAD entry

enum { MQ_OP_A = 0, MQ_OP_U = 1, MQ_OP_L = 2, MQ_OP_LMU = 3 };
enum { MQ_SLOT_LINE = 0, MQ_SLOT_INS = 1 };
// scalar-factor kinds in a family header (index into the per-point scalar arrays of the piece)
enum { MQ_SC_R = 0, MQ_SC_AT = 1, MQ_SC_AQ = 2 };

struct DevSlot {
  int8_t kind;    // MQ_SLOT_LINE / MQ_SLOT_INS
  int8_t zline;   // line index of z for a line slot; for an insertion the line before it (routing only)
  int8_t sgn;     // -1 before the external vertex, +1 after (A' only)
  int8_t child;   // child index for an insertion, else -1
  uint32_t eps;   // bit i: own chord i spans this slot
};

struct DevGeom {
  int32_t nch, nslot, nchild, nS;         // own chords, momentum slots, children, S-type children
  int32_t chord_zline[MQ_MAXL];           // photon line index of own chord i
  DevSlot slot[MQ_MAXSLOT];
  int8_t child_type[MQ_MAXCHILD];         // 0 = S, 1 = V
  int8_t child_patbit[MQ_MAXCHILD];       // bit position of an S-child in the compressed pattern, -1 for V
  int16_t pad;
  int32_t first_table, ntable;            // tables of this geom are consecutive
  // per-point scalar array S of this piece: r_t at [0,nslot); A_t at off_at (only pieces with insertions, else -1);
  // A'_t/g_t at off_aq (only pieces evaluated under operator A, else -1); beta~_tu (t<u, triangular) at off_bt
  int32_t off_at, off_aq, off_bt, scal_len;
};

struct DevTable {
  int32_t geom, op, nout, nfam;           // nfam = stream ENTRIES of this table (each holds MQ_WL families)
  int32_t first_node, nnode;              // nodes using this table are consecutive
  int64_t stream_off, stream_words;       // in 8-byte words from the blob start
  int64_t n_monomials;                    // stored (dense) numerator coefficients
};

struct DevNode {
  int32_t table, geom, nchild, nout;
  int32_t child[MQ_MAXCHILD];
  int32_t val_off;                        // offset (doubles) of this node's graded value(s) in the per-point array
  int32_t ngr;                            // grades stored per output
};

struct DevTerm { int32_t root, sign; };

struct DevHeader {
  int32_t L, M, diag_id, ngeom, ntable, nnode, nterm, nodeval_len;
  int32_t max_scal_len, wl;               // wl = MQ_WL the streams were laid out for
  double C, cond_max;
  int64_t off_Z, off_invdeg, off_geom, off_table, off_node, off_term, total_words;
  int64_t off_stream, stream_chunks;      // the family streams: stream_chunks chunks of MQ_CHUNK_WORDS words
  int32_t rng, pad0;                      // 0 = Philox4x32-10, 1 = MRG32k3a (mc_options.flags bit 2)
  int64_t off_mrg;                        // rng = 1: [2][64][9] uint32, the powers A^(2^k) mod m of the two companion matrices (row-major)
  // defensive mixture (mc_options.mix_alpha > 0; S5b): the second channel's Z, 1/Deg and normalisation, and Deg of BOTH
  // channels (the density of the channel that did not draw the point needs t^Deg_other); all arrays 2^M doubles
  double mix_alpha, C2;
  int64_t off_Z2, off_invdeg2, off_deg1, off_deg2;
};

// Stream entry = MQ_WL families of the SAME shape (c, kd), evaluated side by side by the MQ_WL lanes that share a
// sample point (each lane runs the same static code on its own family; a table with an odd number of families of a
// shape gets a VOID member: zero coefficients). Layout in 8-byte words:
//   hd[MQ_WL] | idx[MQ_WL][idx_words] | coefficients, interleaved
// Family header word hd[s] (uint64):
//   bits  0..2  c   (#Wick pairs; 7 = PAD entry: ONE word, skip 1+idx_words words, no coefficients)      bits  3..5  kd (#inner binary slots)
//   bits  6..9  pattern (compressed)           bits 10..13 nscal (#extra scalar factors)
//   bits 14     out (0/1: which output of an S-type piece)                  bit 15  VOID member
//   bits 16..31 idx_words: 8-byte words of index bytes PER MEMBER
//   bits 32..47 number of coefficient doubles of the WHOLE entry (MQ_WL x per family)
//   bits 48..63 run length: entries from this one to the end of its run of equal shape (c, kd) within the table (>= 1)
//   (c, kd, idx_words and the coefficient count are the same in all MQ_WL header words)
// index bytes of member s: C(2c,2) beta~ indices of its paired slots (pair (i<j) at i*2c - i(i+1)/2 + j-i-1) | kd inner
//   binary slot ids | nscal scalar-factor indices; all are direct indices into the per-point scalar array S
// coefficients: for every pairing (canonical order) 2^kd values per member (index bit b <-> inner slot b). 1 <= kd <= 4:
//   stored as 16-byte units (c[j], c[j+2^(kd-1)]), j < 2^(kd-1) (the first Horner level). kd = 5, 6: the 2^(kd-4) sub-blocks
//   of kd = 4 (top index bits fixed, ascending) one after the other, each in that unit layout. Unit u of a member's
//   Every kd >= 3 block is closed by one more unit (sum_sigma |c_sigma|, 0): the evaluator needs it for a round-off bound that
//   sees the cancellation INSIDE a block (O8); for kd <= 2 it adds the |c| it has loaded anyway. Unit u of a member's sequence sits at unit index u*MQ_WL + s.
//   kd = 0: one double per pairing, at double index q*MQ_WL + s.
//   The lanes of a warp therefore read MQ_WL adjacent units with one shared-memory wavefront.
static inline uint64_t mq_pack_family(int c, int kd, int pattern, int nscal, int out, int idx_words, uint32_t ncoef, int is_void = 0) {
  return (uint64_t)c | (uint64_t)kd << 3 | (uint64_t)pattern << 6 | (uint64_t)nscal << 10 | (uint64_t)out << 14 | (uint64_t)is_void << 15 |
         (uint64_t)idx_words << 16 | (uint64_t)ncoef << 32;
}

// ---- prepare-time path counting (coef_gen.hpp on the host, prep_kernel.cu on the device) ----
enum { MQ_W_FIX = 0, MQ_W_OPEN = 1, MQ_W_CLOSE = 2, MQ_W_BIN = 3, MQ_W_G0 = 4 };
struct MqWElem { uint8_t type, arg; };
// One counting unit: the gamma string of one (slot roles, pairing, functional variant) walked from one start spinor.
// counts[off + 2*sigma + {0,1}] receive the signed number of closed paths with phase (+-1, +-i) per P+/P- pattern sigma.
struct MqCountUnit {
  uint8_t n, start, npairs, pad;
  uint32_t nsig;
  uint64_t off;
  MqWElem el[36];
};
