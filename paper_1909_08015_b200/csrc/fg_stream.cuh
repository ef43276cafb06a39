// fg_stream.cuh — a6 of the double-precision pass: the numerator record stream of one program, run by a block of
// FG_ST_THREADS threads over a batch of FG_ST_SAMPLES samples whose operand tables V (beta, A, A^q) sit in shared memory
// (DESIGN.md "kernels").  Tensor-core groups (FG_REC_MMA, fg_tables.h) are a dense contraction
//   Q[sample][record] = sum_J mono_J[sample] * coef[J][record]
// done with DMMA m8n8k4 (8 samples x 4 monomials x 8 records); sm_100a has no other FP64 tensor shape (the m16n8k4/k8/k16
// f64 shapes of PTX lower to sequences of DMMA.8x8x4 here) and tcgen05 has no FP64 kind.
//
// Work split: warp w serves the 32 samples of sample group sg = w % 8 and the row blocks (8 samples each)
// rb0 .. rb0 + FG_ST_NRB - 1 with rb0 = FG_ST_NRB * (w / 8); two warps share a sample group, so sixteen warps (four per
// scheduler) stream the same tiles in step.  For one row block the monomials of a group are built ONCE (A fragments stay in
// registers for all tiles of the group; the two row blocks of a warp are interleaved column by column so that one 16-byte
// load serves both); per tile the lane loads its B fragment (one conflict-free LDS.32 per k-step: the
// high word of the double), runs the k-steps, and weights its two record values with their products of beta's.
#pragma once
#include "fg_core.cuh"

namespace fg {

#ifndef FG_KO
#define FG_KO 0      // knock-out experiments (timing only, results wrong): 1 no record epilogue, 2 no B loads, 4 no DMMA
#endif
#define FG_ST_THREADS 512
#define FG_ST_SAMPLES 256
#define FG_ST_NRB 2
#define FG_ST_VS (FG_ST_SAMPLES + FG_VPAD)     // row stride of the operand table V (doubles)

__device__ __forceinline__ void dmma884(double& d0, double& d1, double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};" : "+d"(d0), "+d"(d1) : "d"(a), "d"(b));
}

// A (8 samples x 4 monomials): lane (r = lane/4, c = lane%4) holds monomial 4*step + c of sample 8*b + r;
// B (4 monomials x 8 records): lane holds coef[4*step + c] of record r;
// D (8 x 8): lane holds records 2c, 2c+1 of sample 8*b + r.
// The FG_ST_NRB row blocks of the warp go through a tile together: one B fragment and one decoded record header serve
// them all (shared-memory wavefronts, not the FP64 pipe, are what this loop has to economise: ncu, profiles/).
// part[bi] += value partial, part[FG_ST_NRB + bi] += |.| partial of row block rb0 + bi (reduced over the quad by fold_parts).
// partial sums travel by value (registers): a pointer into the caller's state would pin that state to local memory
struct MmaPart { double v[2 * FG_ST_NRB]; };
struct AccPair { double acc, aab; };
template <int NF, int K, bool QX>
__device__ __noinline__ AccPair run_group_static_v(const unsigned char* __restrict__ p, int nrec, const double* __restrict__ Vt, int vs, int ne, AccPair in, int r0) {
  double a = in.acc, b = in.aab;
  run_group_static_body<double, 1, 1, NF, K, QX>(p, nrec, Vt, vs, ne, &a, &b, r0);
  AccPair out; out.acc = a; out.aab = b; return out;
}

// VAR (k = 4 only): 0 every step, 1 / 2 the steps of set A / B of a group flagged FG_REC_PAR_A / FG_REC_PAR_B
template <int NF, int K, bool QX, int VAR = 0>
__device__ __noinline__ MmaPart run_group_mma_rb(const unsigned char* __restrict__ p, int nseq, const double* __restrict__ Vw, int ne, int rb0, MmaPart part) {
  __builtin_assume(__isShared(p)); __builtin_assume(__isShared(Vw));
  constexpr int NM = K < 2 ? 1 : 1 << (K - 2), STEPS = mma_steps(K, QX), TILE = FG_TILE_BYTES(STEPS), NRB = FG_ST_NRB;
  constexpr bool PAR4 = K == 4 && VAR != 0;           // flagged groups: parity-homogeneous step order (fg_tables.h)
  constexpr unsigned SMASK = VAR == 1 ? FG_MMA_PAR_MASK_A(QX) : VAR == 2 ? FG_MMA_PAR_MASK_B(QX) : (1u << STEPS) - 1u;   // steps that are run
  constexpr int ROWB = FG_ST_VS * 8;                 // bytes of one row of V
  const int lane = threadIdx.x & 31, r = lane >> 2, c = lane & 3;
  const int vq = ne * ROWB;
  static_assert(FG_ST_NRB == 2, "the two row blocks of a warp are interleaved column by column");
  // columns: row r of row block rb0 + bi is column 8 * rb0 + 2 * r + bi of the warp's sample group, so that one 16-byte load
  // serves both row blocks (the DMMA does not care which sample sits in which row; fold_parts uses the same map)
  const unsigned char* __restrict__ Vb = (const unsigned char*)(Vw + 8 * rb0 + 2 * r);
  // the lane's base address goes through an opaque asm: ptxas otherwise rebuilds it from %tid (S2R + four integer
  // instructions) in front of every load of the record epilogue to save one register (+11-17 % samples/s, A/B in profiles/)
  { uint32_t vb32 = (uint32_t)__cvta_generic_to_shared(Vb); asm volatile("" : "+r"(vb32)); Vb = (const unsigned char*)__cvta_shared_to_generic(vb32); __builtin_assume(__isShared(Vb)); }
  double av[NRB], ab[NRB];
#pragma unroll
  for (int bi = 0; bi < NRB; ++bi) { av[bi] = part.v[bi]; ab[bi] = part.v[NRB + bi]; }
  for (int g = 0; g < nseq; ++g) {       // consecutive groups of this class (same destination), each with its own free variables
    const uint4 gw = *(const uint4*)p; p += sizeof(FgGroupHdr);
    const int ntiles = (int)(gw.x & 0xffffu);
    const int v0 = (int)((gw.y >> 16) & 255u) * ROWB, v1 = (int)(gw.y >> 24) * ROWB, v2 = (int)(gw.z & 255u) * ROWB, v3 = (int)((gw.z >> 8) & 255u) * ROWB;
    // the lane's column of the A fragments of every k-step (monomial order: fg_tables.h, mma_monomials), built once per group
    double mono[NRB][STEPS];
    if constexpr (K < 2) {       // one step {1, a0, aq0, 0}[c]
      double2 A0 = make_double2(0.0, 0.0), Q0 = make_double2(0.0, 0.0);
      if (K == 1) { A0 = *(const double2*)(Vb + v0); if (QX) Q0 = *(const double2*)(Vb + v0 + vq); }
      mono[0][0] = (c == 0) ? 1.0 : (c == 1) ? A0.x : (c == 2) ? Q0.x : 0.0;
      mono[1][0] = (c == 0) ? 1.0 : (c == 1) ? A0.y : (c == 2) ? Q0.y : 0.0;
    } else {
      const double2 A0 = *(const double2*)(Vb + v0), A1 = *(const double2*)(Vb + v1);
      double2 A2 = make_double2(1.0, 1.0), A3 = make_double2(1.0, 1.0), Q0, Q1, Q2, Q3;
      if (K > 2) A2 = *(const double2*)(Vb + v2);
      if (K > 3) A3 = *(const double2*)(Vb + v3);
      if (QX) { Q0 = *(const double2*)(Vb + v0 + vq); Q1 = *(const double2*)(Vb + v1 + vq); if (K > 2) Q2 = *(const double2*)(Vb + v2 + vq); if (K > 3) Q3 = *(const double2*)(Vb + v3 + vq); }
#pragma unroll
      for (int bi = 0; bi < NRB; ++bi) {
        const double a0 = bi ? A0.y : A0.x, a1 = bi ? A1.y : A1.x, a2 = bi ? A2.y : A2.x, a3 = bi ? A3.y : A3.x;
        if (PAR4) {       // monomial order of k = 4: fg_tables.h (LO/HI pairs by parity; q steps = (j, parity) over the other three)
          const bool c1 = (c & 1) != 0, c2 = (c & 2) != 0;
          const double p01 = a0 * a1, p23 = a2 * a3;
          const double lo0 = c1 ? p01 : 1.0, lo1 = c1 ? a1 : a0, hi0 = c2 ? p23 : 1.0, hi1 = c2 ? a3 : a2;
          mono[bi][0] = lo0 * hi0; mono[bi][1] = lo1 * hi0; mono[bi][2] = lo0 * hi1; mono[bi][3] = lo1 * hi1;
          if (QX) {
            const double q0 = bi ? Q0.y : Q0.x, q1 = bi ? Q1.y : Q1.x, q2 = bi ? Q2.y : Q2.x, q3 = bi ? Q3.y : Q3.x;
            const double p02 = a0 * a2, p03 = a0 * a3, p12 = a1 * a2, p13 = a1 * a3;
            // even: {1, r0 r1, r0 r2, r1 r2}[c], odd: {r0 r1 r2, r2, r1, r0}[c] for (r0, r1, r2) = the variables other than j
#define FG_EO(r0_, r1_, r2_, p01_, p02_, p12_, ev, od) \
            const double ev = (c == 0) ? 1.0 : (c == 1) ? p01_ : (c == 2) ? p02_ : p12_; \
            const double od = (c == 0) ? p01_ * r2_ : (c == 1) ? r2_ : (c == 2) ? r1_ : r0_;
            FG_EO(a1, a2, a3, p12, p13, p23, e0, o0) FG_EO(a0, a2, a3, p02, p03, p23, e1, o1)
            FG_EO(a0, a1, a3, p01, p03, p13, e2, o2) FG_EO(a0, a1, a2, p01, p02, p12, e3, o3)
#undef FG_EO
            mono[bi][4] = q0 * e0; mono[bi][5] = q0 * o0; mono[bi][6] = q1 * e1; mono[bi][7] = q1 * o1;
            mono[bi][8] = q2 * e2; mono[bi][9] = q2 * o2; mono[bi][10] = q3 * e3; mono[bi][11] = q3 * o3;
          }
          continue;
        }
        const double a01 = a0 * a1;
        const double mlo = (c & 2) ? ((c & 1) ? a01 : a1) : ((c & 1) ? a0 : 1.0);
        double hi[NM]; hi[0] = 1.0;
        if (K > 2) hi[1] = a2;
        if (K > 3) { hi[2] = a3; hi[3] = a2 * a3; }
        mono[bi][0] = mlo;
#pragma unroll
        for (int tt = 1; tt < NM; ++tt) mono[bi][tt] = mlo * hi[tt];
        if (QX) {
          const double q0 = bi ? Q0.y : Q0.x, q1 = bi ? Q1.y : Q1.x;
          const double mq = ((c & 2) ? q1 : q0) * ((c & 1) ? ((c & 2) ? a0 : a1) : 1.0);
          mono[bi][NM] = mq;
#pragma unroll
          for (int tt = 1; tt < NM; ++tt) mono[bi][NM + tt] = mq * hi[tt];
          if (K == 3) mono[bi][2 * NM] = mlo * (bi ? Q2.y : Q2.x);
          if (K == 4) {
            const double m2 = mlo * (bi ? Q2.y : Q2.x), m3 = mlo * (bi ? Q3.y : Q3.x);
            mono[bi][2 * NM] = m2; mono[bi][2 * NM + 1] = m2 * a3; mono[bi][2 * NM + 2] = m3; mono[bi][2 * NM + 3] = m3 * a2;
          }
        }
      }
    }
    double pf[NRB][NF > 0 ? NF : 1];
#pragma unroll
    for (int bi = 0; bi < NRB; ++bi) for (int i = 0; i < (NF > 0 ? NF : 1); ++i) pf[bi][i] = 1.0;
    const unsigned char* __restrict__ pt = p;
    for (int t = 0; t < ntiles; ++t, pt += TILE) {
      const int* __restrict__ Bp = (const int*)(pt + 8 * sizeof(FgRecM)) + lane;
      const uint4 hh = *(const uint4*)(pt + c * 16);                 // headers of the lane's records 2c, 2c+1
      double d[NRB][2];
#pragma unroll
      for (int bi = 0; bi < NRB; ++bi) { d[bi][0] = 0.0; d[bi][1] = 0.0; }
#pragma unroll
      for (int st = 0; st < STEPS; ++st) {
        if (!((SMASK >> st) & 1u)) continue;                         // (compile time) no record of this group has a coefficient in this step
#if FG_KO & 2
        const double b = __hiloint2double(lane + st, 0);
#else
        const double b = __hiloint2double(Bp[st * 32], 0);
#endif
#pragma unroll
        for (int bi = 0; bi < NRB; ++bi) {
#if FG_KO & 4
          d[bi][0] = fma(mono[bi][st], b, d[bi][0]);
#else
          dmma884(d[bi][0], d[bi][1], mono[bi][st], b);
#endif
        }
      }
      // products of beta's of this lane's two records (the lane's depth-first stretch: the prefix stack survives from
      // record to record within the group); the header is decoded once for all row blocks
#if FG_KO & 1
      for (int bi = 0; bi < NRB; ++bi) { av[bi] += d[bi][0] + d[bi][1]; ab[bi] += (double)hh.x; }
#else
#pragma unroll
      for (int e = 0; e < 2; ++e) {
        const uint32_t w0 = e ? hh.z : hh.x, w1 = e ? hh.w : hh.y;
        const double cab = fg_cab16_value(w1 >> 16);
        if (NF > 0) {
          const int keep = (int)((w1 >> 8) & 255u);
#pragma unroll
          for (int i = 0; i < NF; ++i) if (i >= keep) {
            const int off = (int)__byte_perm(i < 4 ? w0 : w1, 0u, 0x4440 + (i & 3)) * ROWB;
            const double2 v = *(const double2*)(Vb + off);
            pf[0][i] = (i == 0) ? v.x : pf[0][i > 0 ? i - 1 : 0] * v.x;
            pf[1][i] = (i == 0) ? v.y : pf[1][i > 0 ? i - 1 : 0] * v.y;
          }
        }
#pragma unroll
        for (int bi = 0; bi < NRB; ++bi) {
          const double bp = NF > 0 ? pf[bi][NF > 0 ? NF - 1 : 0] : 1.0;
          av[bi] = fma(bp, d[bi][e], av[bi]); ab[bi] = fma(fabs(bp), cab, ab[bi]);
        }
      }
#endif
    }
    p += (size_t)ntiles * TILE;
  }
#pragma unroll
  for (int bi = 0; bi < NRB; ++bi) { part.v[bi] = av[bi]; part.v[NRB + bi] = ab[bi]; }
  return part;
}

// Running state of one program in the stream kernel.  acc/aab: accumulators of the current destination (owner threads:
// thread t < FG_ST_SAMPLES owns sample t of the batch); part: per-lane tensor-core partial sums (all threads).
struct StreamState {
  double acc[2], aab[2]; MmaPart part; int cur, has_part, has_half, has_two;
#ifdef FG_PHASE_PROF
  long long* prof; long long tlast;
#endif
};

// Hand the partial sums to the owner threads.  Tensor-core groups: quad-reduce, lane c == 0 of quad r posts the sums of sample
// 32*sg + 8*b + r.  Scalar groups: the helper thread t + 256 (which ran the second half of the records of every scalar group
// on the operands of sample t) posts its accumulators.  The owner adds both.  Block-uniform (every warp walks the same
// stream), two pair barriers (four if two-component records were met); called when the destination changes and at the
// end of a program.  xbuf: [0, 512) tensor-core pairs, [512, 1024) helper pairs.
#ifndef FG_DECOUPLE
#define FG_DECOUPLE 1     // 1: warp pairs (w, w + 8) synchronise among themselves, chunk buffers are released by a counter (A/B: 0 = block barriers)
#endif
// Everything fold_parts exchanges stays inside a warp pair (w, w + 8): both serve sample group w % 8 (tensor-core partial
// sums of its 32 samples; helper thread t + 256 mirrors owner t).  A named barrier per pair therefore replaces the
// block barrier, and the eight pairs drift apart within the slack of the chunk ring: while one pair is in a group
// prologue or a record epilogue another keeps the FP64 pipe busy.
__device__ __forceinline__ void pair_sync() {
#if FG_DECOUPLE
  asm volatile("bar.sync %0, 64;" ::"r"(1 + (int)((threadIdx.x >> 5) & 7)) : "memory");
#else
  __syncthreads();
#endif
}
__device__ __forceinline__ void fold_parts(StreamState& st, double* __restrict__ xbuf) {
  if (!st.has_part && !st.has_half) return;
  const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5, sg = w & 7, rb0 = FG_ST_NRB * (w >> 3);
  const bool owner = tid < FG_ST_SAMPLES;
  if (st.has_part) {
#pragma unroll
    for (int bi = 0; bi < FG_ST_NRB; ++bi) {
      double v = st.part.v[bi], a = st.part.v[FG_ST_NRB + bi];
      v += __shfl_xor_sync(0xffffffffu, v, 1); a += __shfl_xor_sync(0xffffffffu, a, 1);
      v += __shfl_xor_sync(0xffffffffu, v, 2); a += __shfl_xor_sync(0xffffffffu, a, 2);
      if ((lane & 3) == 0) { const int smp = 32 * sg + 8 * rb0 + 2 * (lane >> 2) + bi; xbuf[2 * smp] = v; xbuf[2 * smp + 1] = a; }      // column map of run_group_mma_rb
      st.part.v[bi] = 0.0; st.part.v[FG_ST_NRB + bi] = 0.0;
    }
  }
  if (st.has_half && !owner) { xbuf[2 * FG_ST_SAMPLES + 2 * (tid - FG_ST_SAMPLES)] = st.acc[0]; xbuf[2 * FG_ST_SAMPLES + 2 * (tid - FG_ST_SAMPLES) + 1] = st.aab[0]; }
  pair_sync();
  if (owner) {
    if (st.has_part) { st.acc[0] += xbuf[2 * tid]; st.aab[0] += xbuf[2 * tid + 1]; }
    if (st.has_half) { st.acc[0] += xbuf[2 * FG_ST_SAMPLES + 2 * tid]; st.aab[0] += xbuf[2 * FG_ST_SAMPLES + 2 * tid + 1]; }
  }
  pair_sync();
  if (st.has_two) {        // second component of self-energy elements
    if (!owner) { xbuf[2 * (tid - FG_ST_SAMPLES)] = st.acc[1]; xbuf[2 * (tid - FG_ST_SAMPLES) + 1] = st.aab[1]; }
    pair_sync();
    if (owner) { st.acc[1] += xbuf[2 * tid]; st.aab[1] += xbuf[2 * tid + 1]; }
    pair_sync();
  }
  if (!owner) { st.acc[0] = st.acc[1] = 0.0; st.aab[0] = st.aab[1] = 0.0; }
  st.has_part = 0; st.has_half = 0; st.has_two = 0;
}

// All groups of one chunk.  V: operand table of the batch (row stride vs); owner threads flush finished destinations.
template <class Flush>
__device__ __forceinline__ void run_chunk_s(const unsigned char* __restrict__ chunk, const double* __restrict__ V, int vs, int ne, StreamState& st, double* xbuf, Flush&& flush) {
  __builtin_assume(__isShared(chunk)); __builtin_assume(__isShared(V));
  const int tid = threadIdx.x, w = tid >> 5;
  const bool owner = tid < FG_ST_SAMPLES;
  const double* Vt = V + (tid & (FG_ST_SAMPLES - 1));            // the owner's column; a helper thread mirrors sample tid - 256
  { uint32_t a32 = (uint32_t)__cvta_generic_to_shared(Vt); asm volatile("" : "+r"(a32)); Vt = (const double*)__cvta_shared_to_generic(a32); __builtin_assume(__isShared(Vt)); }
  const double* Vw = V + 32 * (w & 7); const int rb0 = FG_ST_NRB * (w >> 3);
  const int ngroups = ((const FgChunkHdr*)chunk)->ngroups;
  const unsigned char* p = chunk + sizeof(FgChunkHdr);
  for (int g = 0; g < ngroups; ++g) {
    FG_MARK(st, 8);
    const FgGroupHdr gh = *(const FgGroupHdr*)p; p += sizeof(FgGroupHdr);
    const int nrec = gh.nrec, nf = gh.nf, k = gh.k, flags = gh.flags;
    if ((int)gh.dst != st.cur) {
      fold_parts(st, xbuf);
      if (st.cur >= 0 && owner) flush(st.cur, st.acc, st.aab);
      st.cur = gh.dst; st.acc[0] = st.acc[1] = 0.0; st.aab[0] = st.aab[1] = 0.0;      // (helpers: zeroed by fold_parts already)
    }
    const bool qx = (flags & FG_REC_QEXT) != 0;
    if (flags & FG_REC_MMA) {
      st.has_part = 1;
      // consecutive tensor-core groups of the same class and destination are run by one call (run length and size come
      // from the planner)
      const unsigned char* p0 = p - sizeof(FgGroupHdr); const int nseq = gh.nseq;
      const int var = (flags & FG_REC_PAR_A) ? 1 : (flags & FG_REC_PAR_B) ? 2 : 0;
#define FG_MM(NF, K) case NF * 8 + K: if (qx) st.part = run_group_mma_rb<NF, K, true>(p0, nseq, Vw, ne, rb0, st.part); else st.part = run_group_mma_rb<NF, K, false>(p0, nseq, Vw, ne, rb0, st.part); break;
#define FG_MP(NF, V) case NF * 8 + V: if (qx) st.part = run_group_mma_rb<NF, 4, true, V>(p0, nseq, Vw, ne, rb0, st.part); else st.part = run_group_mma_rb<NF, 4, false, V>(p0, nseq, Vw, ne, rb0, st.part); break;
      if (var) {       // k = 4 groups whose coefficients sit in one of the two parity step sets
        switch (nf * 8 + var) {
          FG_MP(0, 1) FG_MP(0, 2) FG_MP(1, 1) FG_MP(1, 2) FG_MP(2, 1) FG_MP(2, 2) FG_MP(3, 1) FG_MP(3, 2) FG_MP(4, 1) FG_MP(4, 2) FG_MP(5, 1) FG_MP(5, 2)
          default: break;
        }
      } else {
        switch (nf * 8 + k) {
          FG_MM(0, 2) FG_MM(0, 3) FG_MM(0, 4) FG_MM(1, 2) FG_MM(1, 3) FG_MM(1, 4) FG_MM(2, 2) FG_MM(2, 3) FG_MM(2, 4)
          FG_MM(3, 2) FG_MM(3, 3) FG_MM(3, 4) FG_MM(4, 2) FG_MM(4, 3) FG_MM(4, 4) FG_MM(5, 2) FG_MM(5, 3) FG_MM(5, 4)
          FG_MM(0, 0) FG_MM(0, 1) FG_MM(1, 0) FG_MM(1, 1) FG_MM(2, 0) FG_MM(2, 1) FG_MM(3, 0) FG_MM(3, 1) FG_MM(4, 0) FG_MM(4, 1) FG_MM(5, 0) FG_MM(5, 1)
          default: break;      // the planner makes tensor-core groups of these classes only
        }
      }
#undef FG_MM
#undef FG_MP
      FG_MARK(st, k < 2 ? 2 : 9 + (k - 2) * 2 + (qx ? 1 : 0));      // 2: k = 0, 1; 9..14: tensor-core groups by class (k = 2, 3, 4; without / with q-extension)
      p = p0 + (size_t)gh.seq_units * 16; g += nseq - 1; continue;
    }
    const int bytes = nrec * (((flags & FG_REC_WIDE) ? (int)sizeof(FgRecW) : (int)sizeof(FgRecC)) + rec_ncoef(k, flags) * (int)sizeof(double));
    // scalar groups: the owner threads take records [0, half), the helper threads [half, nrec) on the same operands
    const int half = (nrec + 1) >> 1, r0 = owner ? 0 : half, r1 = owner ? half : nrec;
    st.has_half = 1; if (flags & FG_REC_TWO) st.has_two = 1;
    if (r0 < r1) {
      bool done = false;
      if (!(flags & (FG_REC_WIDE | FG_REC_TWO))) {
        done = true;
        AccPair ap; ap.acc = st.acc[0]; ap.aab = st.aab[0];
        switch (nf * 8 + k) {
#define FG_CLS(NF, K) case NF * 8 + K: if (qx) ap = run_group_static_v<NF, K, true>(p, r1, Vt, vs, ne, ap, r0); \
                                        else ap = run_group_static_v<NF, K, false>(p, r1, Vt, vs, ne, ap, r0); break;
          FG_CLS(0, 0) FG_CLS(0, 1) FG_CLS(0, 2) FG_CLS(0, 3) FG_CLS(0, 4)
          FG_CLS(1, 0) FG_CLS(1, 1) FG_CLS(1, 2) FG_CLS(1, 3) FG_CLS(1, 4)
          FG_CLS(2, 0) FG_CLS(2, 1) FG_CLS(2, 2) FG_CLS(2, 3) FG_CLS(2, 4)
          FG_CLS(3, 0) FG_CLS(3, 1) FG_CLS(3, 2) FG_CLS(3, 3) FG_CLS(3, 4)
          FG_CLS(4, 0) FG_CLS(4, 1) FG_CLS(4, 2) FG_CLS(4, 3) FG_CLS(4, 4)
          FG_CLS(5, 0) FG_CLS(5, 1) FG_CLS(5, 2) FG_CLS(5, 3) FG_CLS(5, 4)
#undef FG_CLS
          default: done = false; break;
        }
        st.acc[0] = ap.acc; st.aab[0] = ap.aab;
      }
      if (done) FG_MARK(st, 3);
      else {
        const int stride = ((flags & FG_REC_WIDE) ? (int)sizeof(FgRecW) : (int)sizeof(FgRecC)) + rec_ncoef(k, flags) * (int)sizeof(double);
        RecState<double, 1> rs; rs.acc[0][0] = st.acc[0]; rs.acc[1][0] = st.acc[1]; rs.aab[0][0] = st.aab[0]; rs.aab[1][0] = st.aab[1]; rs.cur = st.cur; rs.split = 0; rs.rr = 0;
        run_group_dyn<double, 1, 1>(p + (size_t)r0 * stride, r1 - r0, nf, k, flags, Vt, vs, ne, rs);
        st.acc[0] = rs.acc[0][0]; st.acc[1] = rs.acc[1][0]; st.aab[0] = rs.aab[0][0]; st.aab[1] = rs.aab[1][0];
        FG_MARK(st, 4);
      }
    }
    p += bytes;
  }
}

}  // namespace fg
