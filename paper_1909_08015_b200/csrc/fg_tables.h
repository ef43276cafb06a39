// fg_tables.h — plain-old-data tables the host planner writes and the sm_100a kernels read.
// Notation follows PAPER.md (arXiv:1909.08015) Sec. II-III and DESIGN.md.
#pragma once
#include <stdint.h>

#define FG_MAXL 5          // loops n <= 5
#define FG_MAXNE 10        // own electron lines of one element <= 2n
#define FG_MAXLINES 15     // 3n
#define FG_MAXM 15         // Feynman variables (3n, or 3n-1 after the merge of PAPER.md:222)
#define FG_NDEG 6          // polynomial in t: degrees 0..5
#define FG_KMAX 4          // free variables of one numerator record (dense 2^k table); further ones are enumerated
#define FG_MAXF 10         // product factors of one record
#ifndef FG_CHUNK_BYTES
#define FG_CHUNK_BYTES 32768  // numerator stream is cut into chunks of this size (records and tiles never straddle)
#endif
#ifndef FG_VPAD
#define FG_VPAD 4          // padding (elements) of the row stride of the operand table V in shared memory: rows i and j fall
                           // into the same banks only if i = j mod 4 (32-byte shift per row)
#endif
#define FG_MAXSE 4         // self-energy children of one element
#define FG_MAXVC 5         // vertexlike children of one element
#define FG_MAXMEM 8        // members of one forest
#define FG_VMAX (FG_MAXNE * (FG_MAXNE + 1) / 2 + 2 * FG_MAXNE)   // beta (upper triangle), A, A^q

// Operators of the forest formula R^new
enum { FG_OP_A = 0, FG_OP_U = 1, FG_OP_L = 2, FG_OP_LMU = 3 };

// Element geometry: forest member S with its children shrunk.
struct FgGeomDev {
  uint8_t ne, l, has_x, pad;
  uint8_t line_e[FG_MAXNE];   // global line id of own electron line q (path order)
  uint8_t line_ph[FG_MAXL];   // global line id of own photon a
  uint8_t eta[FG_MAXNE];      // bit a set: own electron line q lies on loop a
  int8_t xiq[FG_MAXNE];       // -1 before the site of v_x, +1 after, 0 if v_x is not in S
};

// (geometry, operator): one numerator program.  Its raw accumulators are R[sig][comp][deg].
struct FgNumDev {
  int32_t geom, op, ncomp, nse;        // ncomp 2 for self-energy elements (u, v), else 1; nse = # self-energy children
  int32_t chunk_begin, chunk_count;    // range in the chunk stream
  int32_t node_begin, node_count;      // nodes that use this program
};

// Value node: a program together with the complete subtree below it.
struct FgNodeDev {
  int32_t num, ncomp, nse, nvc;
  int32_t se_kid[FG_MAXSE];   // node ids, order = signature bits
  int32_t vc_kid[FG_MAXVC];   // node ids
};

// One (F, G') term of the forest formula.
struct FgTermDev {
  int32_t top;                // node of G
  int32_t sign;               // (-1)^{|F|-1}
  int32_t nmem;
  int32_t geom[FG_MAXMEM];    // geometries of the members (for prod U_S^2 and sum W_S)
};

// Numerator stream.  A chunk (FG_CHUNK_BYTES, 16-byte aligned) holds groups; a group
// holds records of ONE class (nf, k, flags) that add to ONE accumulator dst, so the kernel runs a fully static inner loop
// per class.  One record:
//   plain:        value = prod_{f<nf} V[fidx[f]] * sum_T coef[T] prod_{j in T} V[vidx[j]]        (2^k coefs per component)
//   q-extension:  ... + prod * sum_{j<k} V[vidx[j] + ne] * sum_{T subset vars\j} coefq_j[T] prod_{i in T} V[vidx[i]]
//                 (k further tables of 2^(k-1) coefs: the slot that carries gamma^nu with weight A^q_j)
// keep = number of leading product factors shared with the previous record of the group (prefix products are kept).
// cabs = sum of |coef| (max over components): with |A_j|, |A^q_j| <= 1 it bounds the sum of |terms| of the record.
#define FG_REC_TWO 1       // two components (u, v) of a self-energy element
#define FG_REC_QEXT 2      // q-extension tables follow
#define FG_REC_WIDE 4      // records use the wide header (nf > FG_NFC): generic slow path
#define FG_REC_MMA 8       // tensor-core group: records that share their free variables, stored as 8-record tiles
#define FG_REC_PAR_A 16    // tensor-core group, k = 4: coefficients only in the steps of set A (see below)
#define FG_REC_PAR_B 32    // ... of set B
#define FG_NFC 5           // product factors of a compact record (= Wick pairs, <= n)
#ifndef FG_MMA_MINK
#define FG_MMA_MINK 0      // tensor-core groups only for records with at least this many free variables
#endif
#ifndef FG_MMA_MINREC
#define FG_MMA_MINREC 3    // a run of records with equal free variables becomes a tensor-core group from this length on
#endif
struct alignas(16) FgRecC {   // compact record header, 16 bytes, followed by the coefficient tables (even count of doubles)
  uint8_t keep;
  uint8_t fidx[FG_NFC];
  uint8_t vidx[FG_KMAX];
  uint8_t pad[2];
  float cabs;
};
struct alignas(16) FgRecW {   // wide record header, 32 bytes
  uint8_t keep, pad0[3];
  uint8_t fidx[FG_MAXF];
  uint8_t vidx[FG_KMAX];
  uint8_t pad1[10];
  float cabs;
};
static_assert(sizeof(FgRecC) == 16 && sizeof(FgRecW) == 32, "record header sizes");
// Tensor-core group (FG_REC_MMA): for a fixed set of free variables the record values are a dense contraction
//   Q[sample][record] = sum_J mono_J(a, a^q)[sample] * coef[J][record]
// evaluated with DMMA m8n8k4 (8 samples x 4 monomials x 8 records).  Monomial J = 4*step + x.
// k = 0, 1 (one step): {1, a0, aq0, 0}[x] (whatever of it the class has): long runs of such records (products of beta's
//   times a constant or a linear factor) go through the record epilogue of the tile path instead of the scalar interpreter.
// k = 2, 3, 4:
//   main  steps t < 2^(k-2):        mlo[x] * mhi[t],  mlo = {1, a0, a1, a0 a1}, mhi[t] = prod_{bit i of t} a_{2+i}
//   low-q steps (q-extension):      {aq0, aq0 a1, aq1, aq1 a0}[x] * mhi[t]
//   high-q steps, j = 2..k-1:       aq_j * mlo[x] * (product over the subset t' of the other high variables)
// k = 4, groups flagged FG_REC_PAR_A / FG_REC_PAR_B.  The Dirac traces leave many tables with non-zero coefficients on
// subsets of ONE parity only (main table and/or the q tables).  With a step order in which every step holds monomials of
// one parity class,
//   main  step s = plo + 2 phi:     LO[plo][x & 1] * HI[phi][x >> 1],  LO[0] = {1, a0 a1}, LO[1] = {a0, a1},
//                                   HI[0] = {1, a2 a3}, HI[1] = {a2, a3}
//   q     step 4 + 2 j + par:       aq_j * R[par][x] over the other three variables r0 < r1 < r2,
//                                   R[0] = {1, r0 r1, r0 r2, r1 r2}, R[1] = {r0 r1 r2, r2, r1, r0}
// a run of records that has no non-zero coefficient outside one of the two step sets met in practice,
//   with q-extension:    A = main + odd q steps (0xaaf),  B = main + even q steps (0x55f)
//   without:             A = steps 0, 3 (even subsets, 0x9),  B = steps 1, 2 (odd subsets, 0x6),
// is stored in that order and flagged, and the kernel issues the DMMAs of that set only (a third to a half fewer).  The
// tiles still hold every step, zeros included, so the interpreters of the upper rungs only need the order.
// A tile = 8 x FgRecM (product factors, bound) + steps x 32 FgMmaCoef in B-fragment order (lane = 4*record + x).
// The coefficients of a tile are stored as the HIGH 32-bit word of the double (sign, exponent, 20 mantissa bits): the
// planner makes a tensor-core group only of records whose coefficients have a zero low word (integers below 2^21 times
// powers of two: every coefficient met so far), so the double the kernel rebuilds with one register move is the same
// number; half the stream bytes, twice the tiles per chunk, and no conversion instruction in the inner loop.
// Lane c of a quad weights records 2c, 2c+1 of every tile; the planner deals the records of a run out so that these form
// one contiguous stretch of the depth-first matching order, and keep = leading product factors shared with the lane's
// previous record (prefix products stay in registers).
// The group header carries the free variables (vidx) and nrec = number of tiles.
typedef int32_t FgMmaCoef;
#if defined(__CUDA_ARCH__)
__device__ __forceinline__ double fg_mma_coef_value(FgMmaCoef h) { return __hiloint2double(h, 0); }
#else
static inline double fg_mma_coef_value(FgMmaCoef h) { const uint64_t u = (uint64_t)(uint32_t)h << 32; double d; __builtin_memcpy(&d, &u, 8); return d; }
#endif
static inline bool fg_mma_coef_pack(double c, FgMmaCoef* out) {   // host: false if the low word is not zero
  uint64_t u; __builtin_memcpy(&u, &c, 8); *out = (FgMmaCoef)(uint32_t)(u >> 32); return (u & 0xffffffffull) == 0;
}
#define FG_TILE_BYTES(steps) (8 * (int)sizeof(FgRecM) + (steps) * 32 * (int)sizeof(FgMmaCoef))
#ifndef FG_MMA_PARITY
#define FG_MMA_PARITY 1                                   // (A/B: 0 never sets FG_REC_PAR_A / FG_REC_PAR_B)
#endif
#define FG_MMA_PAR_MASK_A(qx) ((qx) ? 0xaafu : 0x9u)
#define FG_MMA_PAR_MASK_B(qx) ((qx) ? 0x55fu : 0x6u)
// subset (bits = variables) of monomial x of a k = 4 step: main steps (bits 0-3 = a0..a3), q steps (bits 0-2 = r0..r2)
#define FG_MMA4_MAIN_SUBSET(step, x) ((((step) & 1) ? (((x) & 1) ? 2 : 1) : (((x) & 1) ? 3 : 0)) | ((((step) >> 1) ? (((x) >> 1) ? 2 : 1) : (((x) >> 1) ? 3 : 0)) << 2))
#define FG_MMA4_Q_SUBSET(par, x) ((par) ? (7 ^ ((x) == 0 ? 0 : (x) == 1 ? 3 : (x) == 2 ? 5 : 6)) : ((x) == 0 ? 0 : (x) == 1 ? 3 : (x) == 2 ? 5 : 6))
// Record header of a tile, 8 bytes: product factors, shared prefix depth, and cab16 = the top 16 bits of the double
// sum |coef| rounded UP (sign, exponent, 4 mantissa bits: a bound, at most 6 % above the sum).
struct alignas(8) FgRecM { uint8_t fidx[FG_NFC]; uint8_t keep; uint16_t cab16; };
#if defined(__CUDA_ARCH__)
__device__ __forceinline__ double fg_cab16_value(uint32_t c) { return __hiloint2double((int)(c << 16), 0); }
#else
static inline double fg_cab16_value(uint32_t c) { const uint64_t u = (uint64_t)c << 48; double d; __builtin_memcpy(&d, &u, 8); return d; }
#endif
static inline uint16_t fg_cab16_pack(double c) {      // host: smallest representable value >= c (c >= 0)
  uint64_t u; __builtin_memcpy(&u, &c, 8); uint64_t top = u >> 48; if (u & 0xffffffffffffull) ++top; return (uint16_t)top;
}
// Tensor-core groups: grp_units = size of the group's tiles, seq_units = total size (headers included) of the nseq
// consecutive groups of the same class and destination that start here inside this chunk (one kernel call runs them
// all); both in units of 16 bytes.
struct alignas(16) FgGroupHdr { uint16_t nrec; uint8_t nf, k, flags, dst; uint8_t vidx[FG_KMAX]; uint16_t nseq, seq_units, grp_units; };
static_assert(sizeof(FgRecM) == 8 && sizeof(FgGroupHdr) == 16, "group header sizes");
struct alignas(16) FgChunkHdr { int32_t ngroups; int32_t pad[3]; };

#define FG_MRG_JUMPS 59      // sample ids below 2^59 (32 outputs per sample)
// Everything the kernels need, passed by value.
struct FgPlanDev {
  int32_t n, M, nlines, merge_var;    // merge_var: variable holding the two merged lines, or -1
  int32_t ngeom, nnum, nnode, nterm;
  int32_t raw_slots, scratch_slots;   // per-sample scratch doubles: raw accumulators; total
  uint8_t var_line0[FG_MAXM], var_line1[FG_MAXM];   // lines of each variable (line1 = 255 if single)
  const FgGeomDev* geoms;
  const FgNumDev* nums;
  const FgNodeDev* nodes;
  const FgTermDev* terms;
  const int32_t* geom_num_begin;      // nums are sorted by geometry: nums of geom g are [begin[g], begin[g+1])
  const int32_t* geom_voff;           // row offset of the operand table of geom g in the per-batch table of all geometries
  int32_t vtot, vmax;                 // rows of all geometries together; of the largest one
  const unsigned char* chunks;        // nchunk * FG_CHUNK_BYTES
  const uint32_t* chunk_used;         // bytes in use of every chunk (multiple of 16): what the TMA copy moves
  // random numbers
  int32_t rng, rng_pad;               // 0 Philox4x32-10, 1 MRG32k3a
  const uint32_t* mrg_jump;           // MRG32k3a: FG_MRG_JUMPS x 2 matrices A_c^(32 2^j) mod m_c, row-major (18 words per j)
  // density
  const double* Z1;                   // 2^M
  const double* Z3;                   // 2^M
  double C[4], D, lnZfull[4];
  // precision control
  double rel_tol, abs_tol, err_eps;
  double quarter_pow;                 // (-1/4)^n
  double fact[FG_NDEG];               // k!
};
