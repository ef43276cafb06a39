// fg_kernels.cu — sm_100a kernels of the hot path and the C ABI (include/fg.h).
//
// Launches per slab of samples (blocks of samples, deferred higher-precision passes):
//   fg_geom_kernel<L>       a1-a5 for a wave of samples: Philox, Hepp-sector sample + pdf, element geometry (double-double
//                           inside, rounded once) -> operand tables V (beta, A, A^q), U, W per element in HBM;
//   fg_stream_kernel        a6-a10 of the double-precision pass: persistent, one block of 512 threads per SM serves batches
//                           of 256 samples; V of one element comes in by bulk TMA, the numerator record stream runs on the
//                           FP64 tensor path (fg_stream.cuh), then node products, forest sum, round-off estimate, queueing
//                           of ill-conditioned samples, y = I/g in compensated FP64;
//   fg_eval_kernel<dd|qd>   re-evaluates the queued samples in double-double, then quad-double (whole path in one kernel);
//   fg_reduce_kernel        folds the per-block partial sums in a fixed order (deterministic).
// The numerator coefficient stream is block-uniform: it is pulled through a two-stage shared-memory ring with
// 1-D bulk TMA copies (cp.async.bulk + mbarrier) while the FP64 pipe works on the previous chunk.  Per-sample
// operands (beta, A, A^q) live in shared memory, per-sample polynomials in a per-block scratch.
#include <cuda_runtime.h>

#include <cmath>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <string>
#include <vector>

#include "../../include/fg.h"
#include "fg_core.cuh"
#include "fg_plan.hpp"
#include "fg_stream.cuh"

namespace fg {

struct RunArgs {
  uint64_t first, n, seed;
  const uint32_t* idlist; const unsigned long long* idcount;   // work list (ordinals relative to first) or NULL
  const double* zin;                                           // points instead of samples, or NULL
  double *outI, *outId, *outY, *outErr; uint8_t* outFlags;     // optional per-sample dumps, indexed by ordinal
  uint32_t* flag_bits;                                         // one bit per ordinal: queued for the next rung (compacted in id order afterwards)
  int do_flag;
  double* partials;                                            // [gridDim.x][8]
  void* scratch;
  unsigned long long* phase_cycles;                            // [16] profiling build only (FG_PHASE_PROF), else NULL
  // wave of the double-precision pass: ordinals [ord0, ord0 + nb * FG_ST_SAMPLES) of the slab, tables written by fg_geom_kernel
  uint64_t ord0; int nb;
  double* gV;      // [nb][vtot][FG_ST_VS]   operand tables of all element geometries
  double* gUW;     // [nb][2 * ngeom][FG_ST_SAMPLES]
  double* gMisc;   // [nb][FG_GM_ROWS][FG_ST_SAMPLES]: pdf mantissa, pdf exponent, state, z of the merged variable, amax, amp
};
enum { FG_GM_MANT = 0, FG_GM_EX, FG_GM_STATE, FG_GM_ZM, FG_GM_AMAX, FG_GM_AMP, FG_GM_ROWS };

struct Accum { double sy[2], sy2[2]; unsigned long long nflag, nflag2, nrej, nbig, n; };

// ---- mbarrier / bulk-copy helpers (sm_90+ PTX; SASS: UBLKCP, SYNCS) -------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) { asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory"); }
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) { asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory"); }
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
  uint32_t ok;
  do { asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}" : "=r"(ok) : "r"(smem_u32(bar)), "r"(parity) : "memory"); } while (!ok);
}
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, uint32_t bytes, uint64_t* bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(dst)), "l"(src), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}

struct ChunkRing { unsigned char* buf; uint64_t* bar; uint32_t* cnt; uint32_t phase[2];      // cnt: warps that have left each buffer (stream kernel)
#ifdef FG_PHASE_PROF
  long long* prof; long long tlast;
#endif
};

// a6: run the record stream of one program for the S samples of this thread
template <class T, int S, int ABS>
__device__ void run_program(const FgPlanDev& P, const FgNumDev& N, const ScratchMap& sm, ChunkRing& ring, const T* Vt, int vs, int ne, T* Sc, int ss, int split) {
  const int nslots = (1 << N.nse) * FG_NDEG * N.ncomp;
  for (int i = 0; i < nslots; ++i) {
#pragma unroll
    for (int s = 0; s < S; ++s) { Sc[(sm.rawv + i) * ss + s] = T(0.0); if (ABS) Sc[(sm.rawa + i) * ss + s] = T(0.0); }
  }
  const int nch = N.chunk_count;
  if (nch == 0) return;
  const unsigned char* g0 = P.chunks + (size_t)N.chunk_begin * FG_CHUNK_BYTES;
  const uint32_t* used = P.chunk_used + N.chunk_begin;
  if (threadIdx.x == 0) {
    mbar_expect_tx(&ring.bar[0], used[0]); bulk_g2s(ring.buf, g0, used[0], &ring.bar[0]);
    if (nch > 1) { mbar_expect_tx(&ring.bar[1], used[1]); bulk_g2s(ring.buf + FG_CHUNK_BYTES, g0 + FG_CHUNK_BYTES, used[1], &ring.bar[1]); }
  }
  RecState<T, S> st; st.cur = -1; st.split = split; st.rr = 0;
#ifdef FG_PHASE_PROF
  st.prof = ring.prof; st.tlast = ring.tlast;
#endif
  const int nc = N.ncomp, rawv = sm.rawv, rawa = sm.rawa;
  auto flush = [&](int dst, const T (*acc)[S], const double (*aab)[S]) {
    for (int c = 0; c < nc; ++c) {
#pragma unroll
      for (int s = 0; s < S; ++s) { Sc[(rawv + dst * nc + c) * ss + s] = acc[c][s]; if (ABS) Sc[(rawa + dst * nc + c) * ss + s] = T(aab[c][s]); }
    }
  };
  for (int ch = 0; ch < nch; ++ch) {
    const int b = ch & 1;
    mbar_wait(&ring.bar[b], ring.phase[b]); ring.phase[b] ^= 1u;
    FG_MARK(st, 5);
    run_chunk<T, S, ABS>(ring.buf + b * FG_CHUNK_BYTES, Vt, vs, ne, st, flush);
    FG_MARK(st, 8);
    __syncthreads();   // every thread is done with buffer b
    FG_MARK(st, 5);
    if (threadIdx.x == 0 && ch + 2 < nch) { mbar_expect_tx(&ring.bar[b], used[ch + 2]); bulk_g2s(ring.buf + b * FG_CHUNK_BYTES, g0 + (size_t)(ch + 2) * FG_CHUNK_BYTES, used[ch + 2], &ring.bar[b]); }
  }
  if (st.cur >= 0) { fold_split(st); flush(st.cur, st.acc, st.aab); }
  FG_MARK(st, 8);
#ifdef FG_PHASE_PROF
  ring.tlast = st.tlast;
#endif
}

// Precision rungs.  unit: round-off unit of the running error estimate K * u * sum|terms|;
// geom_unit: relative error of the geometry step per unit of its conditioning `amp`.
template <class T> struct prec;
template <> struct prec<double> { static const int rung = 0; static __device__ double unit(double e, double af) { return e * af; } static __device__ double geom_unit() { return 0x1p-109; } };
template <> struct prec<dd> { static const int rung = 1; static __device__ double unit(double e, double) { return e * 0x1p-51; } static __device__ double geom_unit() { return 0x1p-109; } };
template <> struct prec<qd> { static const int rung = 2; static __device__ double unit(double e, double) { return e * 0x1p-147; } static __device__ double geom_unit() { return 0x1p-205; } };

// Extended rungs: the conditioning of the geometry step is MEASURED instead of bounded.  The product of pivot ratios that
// the double rung uses as `amp` is a worst-case bound: up to 2^130 in corners of the simplex where all photon loops share
// the dominant electron lines (B nearly of rank one), although the true amplification is far smaller; with that bound the
// last rung would reject samples whose value is correct to every digit.  For a sample that fails the tolerance with the
// bound, the elimination of every element is run again, in the given loop order and in the REVERSE order.  The loop matrix B is a sum of at most ten doubles per entry, exact in double-double and
// beyond, so all the error of the step comes from the elimination, and the two orders round independently: delta = the
// largest relative difference between the two tables measures it.  Returned in units of geom_unit, with a factor 4; if the
// two runs share fewer than 30 bits the worst-case bound stays.
template <class T>
__device__ __noinline__ double measured_conditioning(const FgPlanDev& P, const double* z) {
  double zl[FG_MAXLINES];
  for (int v = 0; v < P.M; ++v) {
    const int l0 = P.var_line0[v], l1 = P.var_line1[v];
    if (l1 == 255) zl[l0] = z[v]; else { zl[l0] = 0.5 * z[v]; zl[l1] = 0.5 * z[v]; }
  }
  auto rel = [](const T& a, const T& b) { const double d = to_double(a - b), s = t_abs_d(a); return s != 0.0 ? fabs(d) / s : (d != 0.0 ? 1.0 : 0.0); };
  double amp = 1.0;
  for (int g = 0; g < P.ngeom; ++g) {
    const FgGeomDev E = P.geoms[g];
    FgGeomDev R = E;
    for (int a = 0; a < E.l; ++a) R.line_ph[a] = E.line_ph[E.l - 1 - a];
    for (int q = 0; q < E.ne; ++q) { unsigned m = 0; for (int a = 0; a < E.l; ++a) if ((E.eta[q] >> a) & 1u) m |= 1u << (E.l - 1 - a); R.eta[q] = (uint8_t)m; }
    T V1[FG_VMAX], V2[FG_VMAX], U1, W1, U2, W2; double am, bound, cp2;
    geom_eval<T>(E, zl, V1, 1, U1, W1, am, bound);
    geom_eval<T>(R, zl, V2, 1, U2, W2, am, cp2);
    const int nv = E.ne * (E.ne + 1) / 2 + 2 * E.ne;
    double delta = fmax(rel(U1, U2), rel(W1, W2));
    for (int i = 0; i < nv; ++i) delta = fmax(delta, rel(V1[i], V2[i]));
    const double a = (delta <= 0x1p-30) ? 4.0 * fmax(delta / prec<T>::geom_unit(), 1.0) : bound;
    if (a > amp || !(a == a)) amp = a;
  }
  return amp;
}

// a5-a7 for the S points of this thread
template <class T, int S, int ABS>
__device__ void eval_points(const FgPlanDev& P, ChunkRing& ring, const double (*z)[FG_MAXM], T* Vt, int vs, T* Sc, int ss, T* I, double* Iabs, double* amx, double* amp, int split) {
  const ScratchMap sm(P);
  double zl[S][FG_MAXLINES];
#pragma unroll
  for (int s = 0; s < S; ++s) {
    for (int v = 0; v < P.M; ++v) {
      const int l0 = P.var_line0[v], l1 = P.var_line1[v];
      if (l1 == 255) zl[s][l0] = z[s][v]; else { zl[s][l0] = 0.5 * z[s][v]; zl[s][l1] = 0.5 * z[s][v]; }
    }
    amx[s] = 1.0; amp[s] = 1.0;
  }
  for (int g = 0; g < P.ngeom; ++g) {
    const FgGeomDev E = P.geoms[g];
#pragma unroll
    for (int s = 0; s < S; ++s) {
      T U, W; double am, cp;
      geom_eval<T>(E, zl[s], Vt + s, vs, U, W, am, cp);
      Sc[(2 * g) * ss + s] = U; Sc[(2 * g + 1) * ss + s] = W;
      if (am > amx[s] || !(am == am)) amx[s] = am;
      if (cp > amp[s] || !(cp == cp)) amp[s] = cp;
    }
    FG_MARK(ring, 1);
    for (int ni = P.geom_num_begin[g]; ni < P.geom_num_begin[g + 1]; ++ni) {
      const FgNumDev N = P.nums[ni];
      run_program<T, S, ABS>(P, N, sm, ring, Vt, vs, (int)E.ne, Sc, ss, split);
      for (int k = 0; k < N.node_count; ++k) {
#pragma unroll
        for (int s = 0; s < S; ++s) { finish_node<T, false>(P, sm, N.node_begin + k, Sc + s, ss); if (ABS) finish_node<T, true>(P, sm, N.node_begin + k, Sc + s, ss); }
      }
      FG_MARK(ring, 6);
    }
  }
#pragma unroll
  for (int s = 0; s < S; ++s) {
    T Iv, Ia; assemble<T, ABS != 0>(P, sm, Sc + s, ss, Iv, Ia);
    if (P.merge_var >= 0) { Iv = Iv * T(z[s][P.merge_var]); Ia = Ia * T(z[s][P.merge_var]); }
    I[s] = Iv; Iabs[s] = to_double(Ia);
  }
}


// a8-a9 for one sample: round-off estimate against the tolerance, queueing / rejection, y = I/g, compensated sums
struct TailAcc { dd sy, sy2; unsigned long long nflag, nrej, nbig; };
template <class T>
__device__ __forceinline__ void sample_tail(const FgPlanDev& P, const RunArgs& A, T I, double Iabs, double growth, double amp, double mant, int ex, bool bad, uint64_t oid, TailAcc& ta) {
  const double Id = to_double(I);
  double af = growth * growth; af = af * af * af;      // |A|, |A^q| <= 1 is assumed by cabs; amax^6 otherwise
  // running error estimate: K * u * sum|terms| with u = 2^-53 (double pass), 2^-104 (double-double) or 2^-205 (quad-double)
  // plus the conditioning of the geometry step (double-double, or quad-double in the last rung), DESIGN.md "precision"
  const double err = (prec<T>::unit(P.err_eps, af) + amp * prec<T>::geom_unit()) * Iabs;
  uint8_t fl = 0; double y = 0.0;
  if (!A.idlist && (ex > 1023 || ex < -1021)) ++ta.nbig;
  if (bad) { ++ta.nrej; fl = 2; }
  else {
    const double tol = fmax(P.rel_tol * fabs(Id), ldexp(P.abs_tol * mant, ex));
    const bool over = !(err <= tol);
    if (over && A.do_flag) {
      fl = prec<T>::rung == 0 ? 1 : 8; ++ta.nflag;          // queued for the next rung
      if (A.flag_bits) atomicOr(&A.flag_bits[oid >> 5], 1u << (oid & 31u));
    } else if (over && prec<T>::rung > 0) {
      fl = 4; ++ta.nrej;     // not resolved by the last rung: contributes 0 and is counted
    } else {
      const T yq = I / T(mant);
      y = ldexp(to_double(yq), -ex);
      if (!isfinite(y)) { ++ta.nrej; fl |= 2; y = 0.0; }
      else { ta.sy = dd_add_d(ta.sy, y); ta.sy2 = ta.sy2 + two_prod(y, y); }
    }
  }
  if (A.outI) A.outI[oid] = Id;
  if (A.outId && prec<T>::rung == 0) A.outId[oid] = Id;
  if (A.outY) A.outY[oid] = y;
  if (A.outErr && (prec<T>::rung == 0 || !A.idlist)) A.outErr[oid] = err;
  if (A.outFlags) A.outFlags[oid] = prec<T>::rung > 0 ? (uint8_t)(A.outFlags[oid] | fl) : fl;
}

__device__ __forceinline__ dd shfl_dd(dd v, int off) { return dd(__shfl_down_sync(0xffffffffu, v.hi, off), __shfl_down_sync(0xffffffffu, v.lo, off)); }

// a10: warp shuffle -> block -> one partial per block (added to what the block left there in earlier waves of the slab)
__device__ __forceinline__ void block_reduce_tail(TailAcc& ta, double* red /* shared, 8 doubles per warp */, double* partial, int flag_slot) {
  const int tid = threadIdx.x, nw = blockDim.x >> 5;
  double cnt[3] = {(double)ta.nflag, (double)ta.nrej, (double)ta.nbig};
  for (int off = 16; off > 0; off >>= 1) { ta.sy = ta.sy + shfl_dd(ta.sy, off); ta.sy2 = ta.sy2 + shfl_dd(ta.sy2, off); for (int k = 0; k < 3; ++k) cnt[k] += __shfl_down_sync(0xffffffffu, cnt[k], off); }
  __syncthreads();
  if ((tid & 31) == 0) { double* r = red + (tid >> 5) * 8; r[0] = ta.sy.hi; r[1] = ta.sy.lo; r[2] = ta.sy2.hi; r[3] = ta.sy2.lo; r[4] = cnt[0]; r[5] = cnt[1]; r[6] = cnt[2]; }
  __syncthreads();
  if (tid == 0) {
    dd a(partial[0], partial[1]), b(partial[2], partial[3]); double c[3] = {0.0, partial[5], partial[6]};
    for (int w = 0; w < nw; ++w) { const double* r = red + w * 8; a = a + dd(r[0], r[1]); b = b + dd(r[2], r[3]); for (int k = 0; k < 3; ++k) c[k] += r[4 + k]; }
    partial[0] = a.hi; partial[1] = a.lo; partial[2] = b.hi; partial[3] = b.lo; partial[flag_slot] += c[0]; partial[5] = c[1]; partial[6] = c[2];   // slot 4: queued for double-double, 7: for quad-double
  }
}

template <class T, int S, int MAXNT>
__global__ void __launch_bounds__(MAXNT) fg_eval_kernel(const FgPlanDev P, const RunArgs A) {
  const int NT = blockDim.x;
  extern __shared__ __align__(128) unsigned char smem[];
  ChunkRing ring; ring.buf = smem; ring.bar = (uint64_t*)(smem + 2 * FG_CHUNK_BYTES); ring.phase[0] = ring.phase[1] = 0u;
#ifdef FG_PHASE_PROF
  long long prof[9] = {0, 0, 0, 0, 0, 0, 0, 0, 0}; ring.prof = prof; ring.tlast = clock64();
#endif
  T* Vsm = (T*)(smem + 2 * FG_CHUNK_BYTES + 128);
  const int tid = threadIdx.x;
  if (tid == 0) { mbar_init(&ring.bar[0], 1); mbar_init(&ring.bar[1], 1); asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
  __syncthreads();
  const int vs = NT * S + FG_VPAD, ss = NT * S;   // padded row stride of V: rows of different parity fall into different banks
  T* Vt = Vsm + tid * S;
  T* Sc = (T*)A.scratch + (size_t)blockIdx.x * (size_t)P.scratch_slots * ss + tid * S;
  const uint64_t nwork = A.idlist ? (uint64_t)*A.idcount : A.n;
  // short double-double queues: one point per group of w = 2..32 lanes, its records dealt out to the lanes.  A round
  // then takes about 0.115 + 0.885 / w of a round with one point per thread (measured at w = 32: ~7x shorter) and
  // holds 1/w of the points; w minimises rounds x time per round (the same choice in every block)
  int split = 0;
  if (is_ext<T>::value && S == 1 && nwork > 0) {
    const double cap = (double)gridDim.x * NT; double best = ceil((double)nwork / cap);
    for (int w = 2; w <= 32; w <<= 1) { const double c = ceil((double)nwork * w / cap) * (0.115 + 0.885 / w); if (c < best) { best = c; split = w; } }
  }
  const uint64_t per_batch = split ? (uint64_t)(NT / split) : (uint64_t)NT * S, nbatch = (nwork + per_batch - 1) / per_batch;
  TailAcc ta; ta.sy = dd(0.0); ta.sy2 = dd(0.0); ta.nflag = ta.nrej = ta.nbig = 0;
  const int M = P.M;
  for (uint64_t batch = blockIdx.x; batch < nbatch; batch += gridDim.x) {
    double z[S][FG_MAXM], mant[S]; int ex[S]; bool valid[S], bad[S]; uint64_t oid[S];
#pragma unroll
    for (int s = 0; s < S; ++s) {
      const uint64_t ord = split ? batch * per_batch + (uint64_t)(tid / split) : batch * per_batch + (uint64_t)s * NT + tid;
      valid[s] = ord < nwork; bad[s] = false; mant[s] = 0.5; ex[s] = 1; oid[s] = 0;
      if (valid[s]) {
        oid[s] = A.idlist ? (uint64_t)A.idlist[ord] : ord;
        if (A.zin) { for (int v = 0; v < M; ++v) z[s][v] = A.zin[oid[s] * M + v]; }
        else {
          Sample sp; draw_sample(P, P.Z1, P.Z3, A.first + oid[s], A.seed, sp);
          for (int v = 0; v < M; ++v) z[s][v] = sp.z[v];
          mant[s] = sp.mant; ex[s] = sp.ex; bad[s] = sp.bad;
        }
      }
      if (!valid[s] || bad[s]) for (int v = 0; v < M; ++v) z[s][v] = 1.0 / M;
    }
    FG_MARK(ring, 0);
    T I[S]; double Iabs[S], growth[S], amp[S];
    eval_points<T, S, is_ext<T>::value ? 2 : 1>(P, ring, z, Vt, vs, Sc, ss, I, Iabs, growth, amp, split);
#pragma unroll
    for (int s = 0; s < S; ++s) {
      if (!valid[s] || (split && (tid & (split - 1)) != 0)) continue;
      if constexpr (prec<T>::rung >= 1) {       // the bound failed: measure the conditioning of the geometry step instead
        const double Id = to_double(I[s]);
        const double err = (prec<T>::unit(P.err_eps, 1.0) + amp[s] * prec<T>::geom_unit()) * Iabs[s];
        if (!bad[s] && !(err <= fmax(P.rel_tol * fabs(Id), ldexp(P.abs_tol * mant[s], ex[s])))) amp[s] = measured_conditioning<T>(P, z[s]);
      }
      sample_tail<T>(P, A, I[s], Iabs[s], growth[s], amp[s], mant[s], ex[s], bad[s], oid[s], ta);
    }
    FG_MARK(ring, 7);
  }
#ifdef FG_PHASE_PROF
  if (A.phase_cycles && (tid & 31) == 0) for (int k = 0; k < 9; ++k) atomicAdd(&A.phase_cycles[k], (unsigned long long)prof[k]);
#endif
  block_reduce_tail(ta, (double*)smem /* the ring is idle now */, A.partials + (size_t)blockIdx.x * 8, prec<T>::rung == 0 ? 4 : 7);
}

// ---- double-precision pass, first kernel: a1-a5 for one wave of samples ------------------------------------------
// One thread per sample, one block per batch of FG_ST_SAMPLES samples.  Writes, per batch: the operand tables V of every
// element geometry (rows of FG_ST_VS doubles: the row layout of the stream kernel's shared memory, so that one bulk copy
// brings a whole table in), U and W per geometry, and the per-sample record (pdf, state, conditioning).
__global__ void __launch_bounds__(FG_ST_SAMPLES) fg_geom_kernel(const FgPlanDev P, const RunArgs A) {
  const int tid = threadIdx.x, batch = blockIdx.x, M = P.M;
  const uint64_t ord = A.ord0 + (uint64_t)batch * FG_ST_SAMPLES + tid;
  const bool valid = ord < A.n;
  double z[FG_MAXM], mant = 0.5; int ex = 1; bool bad = false;
  if (valid) {
    if (A.zin) { for (int v = 0; v < M; ++v) z[v] = A.zin[ord * M + v]; }
    else {
      Sample sp; draw_sample(P, P.Z1, P.Z3, A.first + ord, A.seed, sp);
      for (int v = 0; v < M; ++v) z[v] = sp.z[v];
      mant = sp.mant; ex = sp.ex; bad = sp.bad;
    }
  }
  if (!valid || bad) for (int v = 0; v < M; ++v) z[v] = 1.0 / M;
  double zl[FG_MAXLINES];
  for (int v = 0; v < M; ++v) {
    const int l0 = P.var_line0[v], l1 = P.var_line1[v];
    if (l1 == 255) zl[l0] = z[v]; else { zl[l0] = 0.5 * z[v]; zl[l1] = 0.5 * z[v]; }
  }
  double amx = 1.0, amp = 1.0;
  double* Vb = A.gV + (size_t)batch * P.vtot * FG_ST_VS + tid;
  double* UWb = A.gUW + (size_t)batch * 2 * P.ngeom * FG_ST_SAMPLES + tid;
  for (int g = 0; g < P.ngeom; ++g) {
    const FgGeomDev E = P.geoms[g];
    double U, W, am, cp;
    geom_eval<double>(E, zl, Vb + (size_t)P.geom_voff[g] * FG_ST_VS, FG_ST_VS, U, W, am, cp);
    UWb[(2 * g) * FG_ST_SAMPLES] = U; UWb[(2 * g + 1) * FG_ST_SAMPLES] = W;
    if (am > amx || !(am == am)) amx = am;
    if (cp > amp || !(cp == cp)) amp = cp;
  }
  double* Mb = A.gMisc + (size_t)batch * FG_GM_ROWS * FG_ST_SAMPLES + tid;
  Mb[FG_GM_MANT * FG_ST_SAMPLES] = mant; Mb[FG_GM_EX * FG_ST_SAMPLES] = (double)ex;
  Mb[FG_GM_STATE * FG_ST_SAMPLES] = !valid ? 2.0 : (bad ? 1.0 : 0.0);
  Mb[FG_GM_ZM * FG_ST_SAMPLES] = P.merge_var >= 0 ? z[P.merge_var] : 1.0;
  Mb[FG_GM_AMAX * FG_ST_SAMPLES] = amx; Mb[FG_GM_AMP * FG_ST_SAMPLES] = amp;
}

// ---- double-precision pass, second kernel: a6-a10 ------------------------------------------------------------------
// shared memory: [ring 2 x FG_CHUNK_BYTES][3 mbarriers, 128 B][exchange buffer 4 x FG_ST_SAMPLES doubles][V: vmax rows]
#define FG_ST_XBUF_BYTES (4 * FG_ST_SAMPLES * 8)
#define FG_ST_SMEM(vmax) (2 * FG_CHUNK_BYTES + 128 + FG_ST_XBUF_BYTES + (size_t)(vmax) * FG_ST_VS * 8)

__device__ void run_program_s(const FgPlanDev& P, const FgNumDev& N, const ScratchMap& sm, ChunkRing& ring, const double* V, int ne, double* Sc, double* xbuf) {
  const int tid = threadIdx.x, ss = FG_ST_SAMPLES; const bool owner = tid < FG_ST_SAMPLES;
  const int nslots = (1 << N.nse) * FG_NDEG * N.ncomp;
  if (owner) for (int i = 0; i < nslots; ++i) { Sc[(sm.rawv + i) * ss] = 0.0; Sc[(sm.rawa + i) * ss] = 0.0; }
  const int nch = N.chunk_count;
  if (nch == 0) return;
  const unsigned char* g0 = P.chunks + (size_t)N.chunk_begin * FG_CHUNK_BYTES;
  const uint32_t* used = P.chunk_used + N.chunk_begin;
#if FG_DECOUPLE
  __syncthreads();      // every warp has left the ring buffers of the previous program
#endif
  if (tid == 0) {
    mbar_expect_tx(&ring.bar[0], used[0]); bulk_g2s(ring.buf, g0, used[0], &ring.bar[0]);
    if (nch > 1) { mbar_expect_tx(&ring.bar[1], used[1]); bulk_g2s(ring.buf + FG_CHUNK_BYTES, g0 + FG_CHUNK_BYTES, used[1], &ring.bar[1]); }
  }
  StreamState st; st.cur = -1; st.has_part = 0; st.has_half = 0; st.has_two = 0; st.acc[0] = st.acc[1] = st.aab[0] = st.aab[1] = 0.0;
#pragma unroll
  for (int i = 0; i < 2 * FG_ST_NRB; ++i) st.part.v[i] = 0.0;
#ifdef FG_PHASE_PROF
  st.prof = ring.prof; st.tlast = ring.tlast;
#endif
  const int nc = N.ncomp, rawv = sm.rawv, rawa = sm.rawa;
  auto flush = [&](int dst, const double* acc, const double* aab) {
    for (int c = 0; c < nc; ++c) { Sc[(rawv + dst * nc + c) * ss] = acc[c]; Sc[(rawa + dst * nc + c) * ss] = aab[c]; }
  };
  for (int ch = 0; ch < nch; ++ch) {
    const int b = ch & 1;
    mbar_wait(&ring.bar[b], ring.phase[b]); ring.phase[b] ^= 1u;
    FG_MARK(st, 5);
    run_chunk_s(ring.buf + b * FG_CHUNK_BYTES, V, FG_ST_VS, ne, st, xbuf, flush);
    FG_MARK(st, 8);
#if FG_DECOUPLE
    // buffer b is released warp by warp: the last of the 16 warps to leave it starts the copy of chunk ch + 2 (the counter
    // only grows; 16 divides 2^32).  No warp waits here; a fast pair runs at most one chunk ahead of the slowest.
    __syncwarp();
    if ((tid & 31) == 0) {
      const uint32_t old = atomicAdd(&ring.cnt[b], 1u);
      if ((old + 1u) % (FG_ST_THREADS / 32) == 0u && ch + 2 < nch) {
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        const uint32_t ub = used[ch + 2];
        mbar_expect_tx(&ring.bar[b], ub); bulk_g2s(ring.buf + b * FG_CHUNK_BYTES, g0 + (size_t)(ch + 2) * FG_CHUNK_BYTES, ub, &ring.bar[b]);
      }
    }
    FG_MARK(st, 5);
#else
    __syncthreads();   // every thread is done with buffer b
    FG_MARK(st, 5);
    if (tid == 0 && ch + 2 < nch) { mbar_expect_tx(&ring.bar[b], used[ch + 2]); bulk_g2s(ring.buf + b * FG_CHUNK_BYTES, g0 + (size_t)(ch + 2) * FG_CHUNK_BYTES, used[ch + 2], &ring.bar[b]); }
#endif
  }
  fold_parts(st, xbuf);
  if (st.cur >= 0 && owner) flush(st.cur, st.acc, st.aab);
  FG_MARK(st, 8);
#ifdef FG_PHASE_PROF
  ring.tlast = st.tlast;
#endif
}

__global__ void __launch_bounds__(FG_ST_THREADS, 1) fg_stream_kernel(const FgPlanDev P, const RunArgs A) {
  extern __shared__ __align__(128) unsigned char smem[];
  ChunkRing ring; ring.buf = smem; ring.bar = (uint64_t*)(smem + 2 * FG_CHUNK_BYTES); ring.phase[0] = ring.phase[1] = 0u;
#ifdef FG_PHASE_PROF
  long long prof[16] = {0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0}; ring.prof = prof; ring.tlast = clock64();
#endif
  uint64_t* barV = ring.bar + 2; uint32_t phaseV = 0u;
  ring.cnt = (uint32_t*)(smem + 2 * FG_CHUNK_BYTES + 64);
  if (threadIdx.x == 0) { ring.cnt[0] = 0u; ring.cnt[1] = 0u; }
  double* xbuf = (double*)(smem + 2 * FG_CHUNK_BYTES + 128);
  double* V = (double*)(smem + 2 * FG_CHUNK_BYTES + 128 + FG_ST_XBUF_BYTES);
  const int tid = threadIdx.x, ss = FG_ST_SAMPLES; const bool owner = tid < FG_ST_SAMPLES;
  if (tid == 0) { mbar_init(&ring.bar[0], 1); mbar_init(&ring.bar[1], 1); mbar_init(barV, 1); asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
  __syncthreads();
  const ScratchMap sm(P);
  double* Sc = (double*)A.scratch + (size_t)blockIdx.x * (size_t)P.scratch_slots * ss + (owner ? tid : 0);
  TailAcc ta; ta.sy = dd(0.0); ta.sy2 = dd(0.0); ta.nflag = ta.nrej = ta.nbig = 0;
  for (int batch = blockIdx.x; batch < A.nb; batch += gridDim.x) {
    double mant = 0.5, zm = 1.0, amx = 1.0, amp = 1.0; int ex = 1, state = 2;
    if (owner) {
      const double* Mb = A.gMisc + (size_t)batch * FG_GM_ROWS * FG_ST_SAMPLES + tid;
      mant = Mb[FG_GM_MANT * FG_ST_SAMPLES]; ex = (int)Mb[FG_GM_EX * FG_ST_SAMPLES]; state = (int)Mb[FG_GM_STATE * FG_ST_SAMPLES];
      zm = Mb[FG_GM_ZM * FG_ST_SAMPLES]; amx = Mb[FG_GM_AMAX * FG_ST_SAMPLES]; amp = Mb[FG_GM_AMP * FG_ST_SAMPLES];
      const double* UWb = A.gUW + (size_t)batch * 2 * P.ngeom * FG_ST_SAMPLES + tid;
      for (int k = 0; k < 2 * P.ngeom; ++k) Sc[k * ss] = UWb[k * FG_ST_SAMPLES];
    }
    FG_MARK(ring, 0);
    for (int g = 0; g < P.ngeom; ++g) {
      const int nv = P.geom_voff[g + 1] - P.geom_voff[g], ne = P.geoms[g].ne;
      __syncthreads();                      // every warp is done with the previous operand table
      if (tid == 0) {
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        const unsigned char* src = (const unsigned char*)(A.gV + ((size_t)batch * P.vtot + P.geom_voff[g]) * FG_ST_VS);
        const uint32_t bytes = (uint32_t)nv * FG_ST_VS * 8u;
        mbar_expect_tx(barV, bytes);
        for (uint32_t o = 0; o < bytes; o += 32768u) bulk_g2s((unsigned char*)V + o, src + o, bytes - o < 32768u ? bytes - o : 32768u, barV);
      }
      mbar_wait(barV, phaseV); phaseV ^= 1u;
      FG_MARK(ring, 1);
      for (int ni = P.geom_num_begin[g]; ni < P.geom_num_begin[g + 1]; ++ni) {
        const FgNumDev N = P.nums[ni];
        run_program_s(P, N, sm, ring, V, ne, Sc, xbuf);
        if (owner) for (int k = 0; k < N.node_count; ++k) { finish_node<double, false>(P, sm, N.node_begin + k, Sc, ss); finish_node<double, true>(P, sm, N.node_begin + k, Sc, ss); }
        FG_MARK(ring, 6);
      }
    }
    if (owner && state != 2) {
      double Iv, Ia; assemble<double, true>(P, sm, Sc, ss, Iv, Ia);
      Iv *= zm; Ia *= zm;
      sample_tail<double>(P, A, Iv, Ia, amx, amp, mant, ex, state == 1, A.ord0 + (uint64_t)batch * FG_ST_SAMPLES + tid, ta);
    }
    FG_MARK(ring, 7);
  }
#ifdef FG_PHASE_PROF
  if (A.phase_cycles && (tid & 31) == 0) for (int k = 0; k < 16; ++k) atomicAdd(&A.phase_cycles[k], (unsigned long long)prof[k]);
#endif
  block_reduce_tail(ta, (double*)smem /* the ring is idle after the block barrier in there */, A.partials + (size_t)blockIdx.x * 8, 4);
}

// Queue of the next rung: the set bits of `bits` as a list of ordinals in ascending order (one block; deterministic, so
// the extended-precision passes add their samples in the same order on every run).
__global__ void __launch_bounds__(1024) fg_compact_kernel(const uint32_t* __restrict__ bits, uint32_t nwords, uint32_t* __restrict__ list, unsigned long long* __restrict__ count) {
  __shared__ uint32_t part[1024];
  const uint32_t t = threadIdx.x, per = (nwords + 1023u) / 1024u, w0 = t * per, w1 = min(nwords, w0 + per);
  uint32_t c = 0;
  for (uint32_t w = w0; w < w1; ++w) c += __popc(bits[w]);
  part[t] = c;
  __syncthreads();
  for (uint32_t off = 1; off < 1024; off <<= 1) {          // inclusive scan
    const uint32_t v = t >= off ? part[t - off] : 0u;
    __syncthreads();
    part[t] += v;
    __syncthreads();
  }
  uint32_t pos = part[t] - c;
  for (uint32_t w = w0; w < w1; ++w) { uint32_t m = bits[w]; while (m) { const int b = __ffs(m) - 1; list[pos++] = w * 32u + (uint32_t)b; m &= m - 1u; } }
  if (t == 1023) *count = (unsigned long long)part[1023];
}

__global__ void fg_reduce_kernel(const double* partials, int nparts, Accum* acc, unsigned long long n_add, int finalize, fg_result* out) {
  if (threadIdx.x != 0 || blockIdx.x != 0) return;
  dd a(acc->sy[0], acc->sy[1]), b(acc->sy2[0], acc->sy2[1]);
  double c[4] = {0, 0, 0, 0};
  for (int i = 0; i < nparts; ++i) { const double* r = partials + (size_t)i * 8; a = a + dd(r[0], r[1]); b = b + dd(r[2], r[3]); for (int k = 0; k < 4; ++k) c[k] += r[4 + k]; }
  acc->sy[0] = a.hi; acc->sy[1] = a.lo; acc->sy2[0] = b.hi; acc->sy2[1] = b.lo;
  acc->nflag += (unsigned long long)c[0]; acc->nrej += (unsigned long long)c[1]; acc->nbig += (unsigned long long)c[2]; acc->nflag2 += (unsigned long long)c[3]; acc->n += n_add;
  if (finalize) {
    const double N = (double)acc->n;
    out->mean = to_double(a) / N;
    const dd v = b / dd(N * N) - a * a / dd(N * N * N);   // (17)
    out->variance = to_double(v);
    out->sum_y[0] = a.hi; out->sum_y[1] = a.lo; out->sum_y2[0] = b.hi; out->sum_y2[1] = b.lo;
    out->n_samples = acc->n; out->n_flagged = acc->nflag; out->n_flagged2 = acc->nflag2; out->n_rejected = acc->nrej; out->n_pdf_big_exp = acc->nbig;
  }
}

__global__ void fg_sample_dump_kernel(const FgPlanDev P, uint64_t first, uint64_t n, uint64_t seed, uint32_t* words, int32_t* comp,
                                      uint8_t* order, double* z, double* mant, int32_t* ex, uint8_t* bad) {
  const uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const uint64_t sid = first + i; const int M = P.M;
  if (words && P.rng == 1) {      // MRG32k3a: the integers (x1 - x2) mod m1 (0 -> m1) of outputs 32 sid, 32 sid + 1, ... (u = integer / (m1 + 1))
    UniformStream us(sid, seed, 1, P.mrg_jump);
    for (int k = 0; k < 4 * M; ++k) words[i * M * 4 + k] = (uint32_t)(us.next_mrg() * 4294967088.0 + 0.5);
  } else
  if (words) for (int c = 0; c < M; ++c) { uint32_t w[4]; philox4x32_10((uint32_t)sid, (uint32_t)(sid >> 32), (uint32_t)c, 0u, (uint32_t)seed, (uint32_t)(seed >> 32), w); for (int k = 0; k < 4; ++k) words[(i * M + c) * 4 + k] = w[k]; }
  Sample sp; draw_sample(P, P.Z1, P.Z3, sid, seed, sp);
  if (comp) comp[i] = sp.comp;
  for (int v = 0; v < M; ++v) { if (order) order[i * M + v] = sp.order[v]; if (z) z[i * M + v] = sp.z[v]; }
  if (mant) mant[i] = sp.mant; if (ex) ex[i] = sp.ex; if (bad) bad[i] = sp.bad ? 1 : 0;
}

// FP64-FMA peak: 8 independent chains per thread (the roofline denominator is measured, not quoted)
__global__ void fg_dfma_kernel(double* out, int iters, double a, double b) {
  double x0 = threadIdx.x * 1e-9, x1 = x0 + 1, x2 = x0 + 2, x3 = x0 + 3, x4 = x0 + 4, x5 = x0 + 5, x6 = x0 + 6, x7 = x0 + 7;
  for (int i = 0; i < iters; ++i) {
    x0 = fma(x0, a, b); x1 = fma(x1, a, b); x2 = fma(x2, a, b); x3 = fma(x3, a, b);
    x4 = fma(x4, a, b); x5 = fma(x5, a, b); x6 = fma(x6, a, b); x7 = fma(x7, a, b);
  }
  out[(size_t)blockIdx.x * blockDim.x + threadIdx.x] = ((x0 + x1) + (x2 + x3)) + ((x4 + x5) + (x6 + x7));
}

// FP64 tensor peak: 8 independent DMMA m8n8k4 accumulator pairs per warp (shares the FP64 units with DFMA)
__global__ void fg_dmma_kernel(double* out, int iters, double a, double b) {
  double c0[8], c1[8];
#pragma unroll
  for (int i = 0; i < 8; ++i) { c0[i] = i + threadIdx.x * 1e-9; c1[i] = -i; }
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int i = 0; i < 8; ++i) asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};" : "+d"(c0[i]), "+d"(c1[i]) : "d"(a), "d"(b));
  }
  double s = 0.0;
#pragma unroll
  for (int i = 0; i < 8; ++i) s += c0[i] + c1[i];
  out[(size_t)blockIdx.x * blockDim.x + threadIdx.x] = s;
}

}  // namespace fg

// =================================================================================================
// C ABI
// =================================================================================================
using namespace fg;

static thread_local std::string g_err;
int fg_internal_fail(int code, const std::string& m) { g_err = m; return code; }     // shared with fg_batch.cpp
static int fail(int code, const std::string& m) { return fg_internal_fail(code, m); }
#define CU(x) do { cudaError_t e_ = (x); if (e_ != cudaSuccess) return fail(FG_E_CUDA, std::string(#x) + ": " + cudaGetErrorString(e_)); } while (0)

struct fg_graph { Graph g; };

#ifndef FG_NT_Q
#define FG_NT_Q 192
#endif
static const int NT_Q = FG_NT_Q, S_Q = 1;     // double-double pass: max threads per block (launch bound), samples per thread
static const int NT_QD = 64;              // quad-double pass
static const uint64_t SLAB = 1ull << 24;  // samples per slab (bounds the re-evaluation queue)
static const size_t WAVE_BYTES = (size_t)3 << 30;   // budget of the operand tables one wave of the double pass keeps in HBM

struct fg_plan {
  HostPlan H; FgPlanDev D; int device = 0, sms = 0;
  std::vector<void*> allocs;
  void* scratch = nullptr; double* partials = nullptr; Accum* accum = nullptr; fg_result* result_dev = nullptr;
  uint32_t* flag_list = nullptr; unsigned long long* flag_count = nullptr; unsigned long long* phase_cycles = nullptr;
  uint32_t* flag_list2 = nullptr; unsigned long long* flag_count2 = nullptr;      // queue of the quad-double rung
  uint32_t *flag_bits = nullptr, *flag_bits2 = nullptr;                           // one bit per sample of the slab, per queue
  int grid_qd = 0, nt_qd = 0; size_t smem_qd = 0;
  int grid_d = 0, grid_q = 0, nt_q = 0; size_t smem_d = 0, smem_q = 0; int vmax = 0;
  int wave_nb = 0; double *gV = nullptr, *gUW = nullptr, *gMisc = nullptr;   // wave buffers of the double pass (fg_geom_kernel -> fg_stream_kernel)
  int64_t table_bytes = 0;
  // per-kernel timing: four events per slab, recorded on the launching stream and resolved later (no host synchronisation
  // inside the timed region); evpool holds the events of the slabs not yet folded into ms[]
  int profile = 0; std::vector<cudaEvent_t> evpool, evfree; double ms[3] = {0, 0, 0}; long long launches = 0;
  std::mutex mu;
};

template <class T> static int upload(fg_plan* p, const std::vector<T>& v, const T** dst) {
  void* d = nullptr; size_t bytes = std::max<size_t>(v.size() * sizeof(T), 16);
  CU(cudaMalloc(&d, bytes)); p->allocs.push_back(d); p->table_bytes += (int64_t)bytes;
  if (!v.empty()) CU(cudaMemcpy(d, v.data(), v.size() * sizeof(T), cudaMemcpyHostToDevice));
  *dst = (const T*)d; return FG_OK;
}

extern "C" {

const char* fg_version(void) { return "fg 0.1 (sm_100a)"; }
const char* fg_last_error_message(void) { return g_err.c_str(); }
const char* fg_strerror(int code) {
  switch (code) {
    case FG_OK: return "ok"; case FG_E_ARG: return "bad argument"; case FG_E_COUNT: return "wrong number of lines or vertices";
    case FG_E_NOT_PATH: return "electron lines are not one open path"; case FG_E_VERTEX: return "vertex without exactly one photon";
    case FG_E_NOT_1PI: return "graph is not one-particle irreducible"; case FG_E_LOOPS: return "more than 5 loops";
    case FG_E_CUDA: return "CUDA error"; case FG_E_LIMIT: return "internal limit exceeded"; case FG_E_OPTS: return "invalid plan options";
    default: return "unknown error";
  }
}

int fg_graph_create(const fg_edge* edges, int32_t n_edges, int32_t ext_photon_vertex, fg_graph** out) {
  if (!out) return fail(FG_E_ARG, "out is NULL");
  *out = nullptr;
  if (!edges) return fail(FG_E_ARG, "edges is NULL");
  fg_graph* G = new fg_graph(); std::string msg;
  int rc = graph_from_edges((const int32_t*)edges, n_edges, ext_photon_vertex, G->g, msg);
  if (rc != FG_OK) { delete G; return fail(rc, msg); }
  *out = G; return FG_OK;
}
void fg_graph_destroy(fg_graph* g) { delete g; }

int fg_graph_class(const fg_graph* g, int32_t* kmm) {      // photons left of / right of / across the external photon
  if (!g || !kmm) return fail(FG_E_ARG, "NULL argument");
  int k = 0, left = 0, right = 0;
  for (auto& ph : g->g.ph) { if (ph[1] < g->g.x) ++left; else if (ph[0] > g->g.x) ++right; else ++k; }
  kmm[0] = k; kmm[1] = left > right ? left : right; kmm[2] = left > right ? right : left;
  return FG_OK;
}

void fg_plan_opts_default(fg_plan_opts* o) {
  if (!o) return;
  std::memset(o, 0, sizeof(*o));
  o->C[0] = 0.9; o->C[1] = 0.03; o->C[2] = 0.01; o->C[3] = 0.06; o->D = 0.75;   // Calc 2
  o->merge_ext_lines = 0; o->deg_table = nullptr; o->rel_tol = 1e-12; o->abs_tol = 0.0; o->err_factor = 0.0;
  o->deg_rule = 0; const double c15[6] = {0.256, 0.839, 0.786, 0.2, 0.0, 0.2};   // eq. (15)
  for (int k = 0; k < 6; ++k) o->deg_consts[k] = c15[k];
}

void fg_plan_destroy(fg_plan* p) {
  if (!p) return;
  cudaSetDevice(p->device);
  for (void* a : p->allocs) cudaFree(a);
  for (cudaEvent_t e : p->evpool) cudaEventDestroy(e);
  for (cudaEvent_t e : p->evfree) cudaEventDestroy(e);
  delete p;
}

int fg_plan_create(const fg_graph* g, const fg_plan_opts* opts, int32_t device, fg_plan** out) {
  if (!out) return fail(FG_E_ARG, "out is NULL");
  *out = nullptr;
  if (!g) return fail(FG_E_ARG, "graph is NULL");
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) return fail(FG_E_CUDA, "no CUDA device: this library has no CPU path");
  if (device < 0 || device >= ndev) return fail(FG_E_ARG, "device out of range");
  fg_plan_opts o; if (opts) o = *opts; else fg_plan_opts_default(&o);
  if (o.deg_rule != 0) return fail(FG_E_OPTS, "deg_rule: only rule 0 is available (the paper's Deg algorithm is in its Refs. [42], [32], PAPER.md:250)");
  if (o.rng != 0 && o.rng != 1) return fail(FG_E_OPTS, "rng: 0 = Philox4x32-10, 1 = MRG32k3a");
  PlanOpts po; for (int k = 0; k < 4; ++k) po.C[k] = o.C[k]; po.D = o.D; po.merge = o.merge_ext_lines ? 1 : 0;
  po.rel_tol = o.rel_tol; po.abs_tol = o.abs_tol; po.err_factor = o.err_factor;
  if (!(po.rel_tol >= 0) || !(po.abs_tol >= 0) || (po.rel_tol == 0 && po.abs_tol == 0)) return fail(FG_E_OPTS, "tolerances: need rel_tol >= 0, abs_tol >= 0, not both 0 (every sample would be rejected)");
  int M = 3 * g->g.n - (po.merge ? 1 : 0);
  if (o.deg_table) po.deg_override.assign(o.deg_table, o.deg_table + ((size_t)1 << M));
  fg_plan* p = new fg_plan(); std::string msg;
  int rc = build_plan(g->g, po, p->H, msg);
  if (rc != FG_OK) { delete p; return fail(rc, msg); }
  p->device = device;
  cudaError_t e = cudaSetDevice(device); if (e != cudaSuccess) { delete p; return fail(FG_E_CUDA, cudaGetErrorString(e)); }
  cudaDeviceProp prop; cudaGetDeviceProperties(&prop, device); p->sms = prop.multiProcessorCount;
  HostPlan& H = p->H; FgPlanDev& D = p->D; std::memset(&D, 0, sizeof(D));
  D.n = H.g.n; D.M = H.M; D.nlines = 3 * H.g.n; D.merge_var = H.merge_var;
  D.ngeom = (int)H.d_geoms.size(); D.nnum = (int)H.d_nums.size(); D.nnode = (int)H.d_nodes.size(); D.nterm = (int)H.d_terms.size();
  D.raw_slots = H.raw_slots; D.scratch_slots = H.scratch_slots;
  for (int v = 0; v < H.M; ++v) { D.var_line0[v] = (uint8_t)H.var_lines[v][0]; D.var_line1[v] = H.var_lines[v].size() > 1 ? (uint8_t)H.var_lines[v][1] : 255; }
  for (int k = 0; k < 4; ++k) { D.C[k] = H.opts.C[k]; D.lnZfull[k] = H.lnZfull[k]; }
  D.D = H.opts.D; D.rel_tol = po.rel_tol; D.abs_tol = po.abs_tol;
  D.err_eps = (po.err_factor > 0 ? po.err_factor : 8.0) * 0x1p-53;
  D.quarter_pow = std::pow(-0.25, H.g.n); D.fact[0] = 1; for (int k = 1; k < FG_NDEG; ++k) D.fact[k] = D.fact[k - 1] * k;
#define UP(vec, field) do { int rc_ = upload(p, vec, &D.field); if (rc_ != FG_OK) { fg_plan_destroy(p); return rc_; } } while (0)
  UP(H.d_geoms, geoms); UP(H.d_nums, nums); UP(H.d_nodes, nodes); UP(H.d_terms, terms); UP(H.d_geom_num_begin, geom_num_begin);
  UP(H.d_chunks, chunks); UP(H.d_chunk_used, chunk_used); UP(H.Z1, Z1); UP(H.Z3, Z3);
  UP(H.d_geom_voff, geom_voff);
  D.rng = o.rng;
  if (o.rng == 1) {      // MRG32k3a: A_c^(32 2^j) mod m_c of the two recurrence matrices, by repeated squaring from A_c^32
    auto mm = [](const uint64_t* a, const uint64_t* b, uint64_t* c, uint64_t m) { uint64_t r[9]; for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) { uint64_t t = 0; for (int k = 0; k < 3; ++k) t = (t + a[3 * i + k] * b[3 * k + j] % m) % m; r[3 * i + j] = t; } for (int i = 0; i < 9; ++i) c[i] = r[i]; };
    const uint64_t m[2] = {FG_MRG_M1, FG_MRG_M2};
    uint64_t B[2][9] = {{0, 1, 0, 0, 0, 1, FG_MRG_M1 - 810728ull, 1403580ull, 0}, {0, 1, 0, 0, 0, 1, FG_MRG_M2 - 1370589ull, 0, 527612ull}};
    for (int c = 0; c < 2; ++c) for (int k = 0; k < 5; ++k) mm(B[c], B[c], B[c], m[c]);      // A^32
    std::vector<uint32_t> jt((size_t)FG_MRG_JUMPS * 18);
    for (int j = 0; j < FG_MRG_JUMPS; ++j) for (int c = 0; c < 2; ++c) { for (int i = 0; i < 9; ++i) jt[(size_t)18 * j + 9 * c + i] = (uint32_t)B[c][i]; mm(B[c], B[c], B[c], m[c]); }
    UP(jt, mrg_jump);
  }
#undef UP
  D.vtot = H.vtot; D.vmax = H.vmax;
  const int vmax = H.vmax; p->vmax = vmax;
  int smem_max = 0; cudaDeviceGetAttribute(&smem_max, cudaDevAttrMaxSharedMemoryPerBlockOptin, device);
  // double pass: one persistent block of FG_ST_THREADS threads per SM, FG_ST_SAMPLES samples per batch
  p->smem_d = FG_ST_SMEM(vmax);
  if ((long)p->smem_d > (long)smem_max) { fg_plan_destroy(p); return fail(FG_E_LIMIT, "element tables do not fit in shared memory"); }
  // double-double pass: as many warps as the per-sample operand table V (vmax entries) leaves room for in shared memory
  const size_t ring_bytes = 2 * FG_CHUNK_BYTES + 128;
  auto fit = [&](int maxnt, size_t per_thread) { long nt = ((long)smem_max - (long)ring_bytes) / (long)per_thread - FG_VPAD; nt = std::min<long>(maxnt, nt / 32 * 32); return (int)nt; };
  // The upper rungs keep run-time-indexed arrays and spills in local memory (7-14 KB of stack per thread); with the whole
  // L1 carved out for shared memory every such access goes to L2 and a round crawls (profiles/r02_dd_kernel_ncu.md).  So a
  // block takes only as many threads as leave ~64 KB of L1 (shared memory <= FG_UPPER_SMEM), but at least 64.
#ifndef FG_UPPER_SMEM
#define FG_UPPER_SMEM (148 * 1024)
#endif
  auto fit_l1 = [&](int nt, size_t per_thread) { long cap = ((long)FG_UPPER_SMEM - (long)ring_bytes) / (long)per_thread - FG_VPAD; cap = std::max<long>(64, cap / 32 * 32); return (int)std::min<long>(nt, cap); };
  p->nt_q = fit_l1(fit(NT_Q, (size_t)vmax * S_Q * sizeof(dd)), (size_t)vmax * S_Q * sizeof(dd));
  if (p->nt_q < 32) { fg_plan_destroy(p); return fail(FG_E_LIMIT, "element tables do not fit in shared memory"); }
  p->smem_q = ring_bytes + (size_t)vmax * (p->nt_q * S_Q + FG_VPAD) * sizeof(dd);
  p->nt_qd = fit(NT_QD, (size_t)vmax * sizeof(qd));
  if (p->nt_qd < 32) { fg_plan_destroy(p); return fail(FG_E_LIMIT, "element tables do not fit in shared memory"); }
  p->smem_qd = ring_bytes + (size_t)vmax * (p->nt_qd + FG_VPAD) * sizeof(qd);
  // the attribute is per function, not per plan: always raise it to the device limit
  auto setattr = [&](const void* f) { return cudaFuncSetAttribute(f, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_max); };
  e = setattr((const void*)fg_stream_kernel); if (e == cudaSuccess) e = setattr((const void*)fg_eval_kernel<dd, S_Q, NT_Q>);
  if (e == cudaSuccess) e = setattr((const void*)fg_eval_kernel<qd, 1, NT_QD>);
  if (e != cudaSuccess) { fg_plan_destroy(p); return fail(FG_E_CUDA, std::string("shared memory: ") + cudaGetErrorString(e)); }
  int bps_q = 1;
  cudaOccupancyMaxActiveBlocksPerMultiprocessor(&bps_q, fg_eval_kernel<dd, S_Q, NT_Q>, p->nt_q, p->smem_q);
  p->grid_d = p->sms; p->grid_q = p->sms * std::max(1, std::min(bps_q, 2)); p->grid_qd = p->sms;
  // a wave = a multiple of the grid in batches, bounded by the HBM budget of its operand tables
  { const size_t per_batch = ((size_t)H.vtot * FG_ST_VS + (size_t)(2 * D.ngeom + FG_GM_ROWS) * FG_ST_SAMPLES) * sizeof(double);
    long rounds = (long)(WAVE_BYTES / (per_batch * (size_t)p->grid_d)); rounds = std::max<long>(1, std::min<long>(rounds, 16));
    p->wave_nb = (int)rounds * p->grid_d; }
  size_t sc = (size_t)H.scratch_slots * std::max(std::max((size_t)FG_ST_SAMPLES * sizeof(double) * p->grid_d, (size_t)p->nt_q * S_Q * sizeof(dd) * p->grid_q), (size_t)p->nt_qd * sizeof(qd) * p->grid_qd);
  auto dmalloc = [&](void** d, size_t bytes) { cudaError_t e2 = cudaMalloc(d, bytes); if (e2 == cudaSuccess) { p->allocs.push_back(*d); cudaMemset(*d, 0, bytes); } return e2; };
  e = dmalloc(&p->scratch, sc);
  if (e == cudaSuccess) e = dmalloc((void**)&p->partials, (size_t)(p->grid_d + p->grid_q + p->grid_qd) * 8 * sizeof(double));
  if (e == cudaSuccess) e = dmalloc((void**)&p->flag_list2, SLAB * sizeof(uint32_t));
  if (e == cudaSuccess) e = dmalloc((void**)&p->flag_bits, SLAB / 8);
  if (e == cudaSuccess) e = dmalloc((void**)&p->flag_bits2, SLAB / 8);
  if (e == cudaSuccess) e = dmalloc((void**)&p->flag_count2, sizeof(unsigned long long));
  if (e == cudaSuccess) e = dmalloc((void**)&p->accum, sizeof(Accum));
  if (e == cudaSuccess) e = dmalloc((void**)&p->result_dev, sizeof(fg_result));
  if (e == cudaSuccess) e = dmalloc((void**)&p->flag_list, SLAB * sizeof(uint32_t));
  if (e == cudaSuccess) e = dmalloc((void**)&p->flag_count, sizeof(unsigned long long));
  if (e == cudaSuccess) e = dmalloc((void**)&p->phase_cycles, 16 * sizeof(unsigned long long));
  if (e == cudaSuccess) e = dmalloc((void**)&p->gV, (size_t)p->wave_nb * H.vtot * FG_ST_VS * sizeof(double));
  if (e == cudaSuccess) e = dmalloc((void**)&p->gUW, (size_t)p->wave_nb * 2 * D.ngeom * FG_ST_SAMPLES * sizeof(double));
  if (e == cudaSuccess) e = dmalloc((void**)&p->gMisc, (size_t)p->wave_nb * FG_GM_ROWS * FG_ST_SAMPLES * sizeof(double));
  if (e != cudaSuccess) { fg_plan_destroy(p); return fail(FG_E_CUDA, std::string("cudaMalloc: ") + cudaGetErrorString(e)); }
  *out = p; return FG_OK;
}

int fg_plan_set_tol(fg_plan* p, double rel_tol, double abs_tol) {
  if (!p || !(rel_tol >= 0) || !(abs_tol >= 0) || (rel_tol == 0 && abs_tol == 0)) return fail(FG_E_ARG, "bad tolerance: need rel_tol >= 0, abs_tol >= 0, not both 0 (every sample would be rejected)");
  std::lock_guard<std::mutex> lk(p->mu);
  p->D.rel_tol = rel_tol; p->D.abs_tol = abs_tol; return FG_OK;
}

// folds the recorded events into ms[] (waits for the last of them)
static int resolve_events(fg_plan* p) {
  for (size_t i = 0; i + 3 < p->evpool.size(); i += 4) {
    CU(cudaEventSynchronize(p->evpool[i + 3]));
    for (int k = 0; k < 3; ++k) { float t = 0; CU(cudaEventElapsedTime(&t, p->evpool[i + k], p->evpool[i + k + 1])); p->ms[k] += t; }
  }
  p->evfree.insert(p->evfree.end(), p->evpool.begin(), p->evpool.end()); p->evpool.clear();
  return FG_OK;
}

int fg_plan_profile(fg_plan* p, int32_t enable) {
  if (!p) return fail(FG_E_ARG, "NULL plan");
  std::lock_guard<std::mutex> lk(p->mu);
  CU(cudaSetDevice(p->device));
  int rc = resolve_events(p); if (rc != FG_OK) return rc;
  p->profile = enable ? 1 : 0; p->ms[0] = p->ms[1] = p->ms[2] = 0; p->launches = 0;
  return FG_OK;
}
int fg_plan_timing(const fg_plan* cp, double* ms3, int64_t* launches) {
  fg_plan* p = const_cast<fg_plan*>(cp);
  if (!p) return fail(FG_E_ARG, "NULL plan");
  std::lock_guard<std::mutex> lk(p->mu);
  CU(cudaSetDevice(p->device));
  int rc = resolve_events(p); if (rc != FG_OK) return rc;
  if (ms3) for (int k = 0; k < 3; ++k) ms3[k] = p->ms[k];
  if (launches) *launches = p->launches;
  return FG_OK;
}

int fg_plan_phase_cycles(const fg_plan* cp, uint64_t* cycles16, int32_t reset) {
  fg_plan* p = const_cast<fg_plan*>(cp);
  if (!p) return fail(FG_E_ARG, "NULL plan");
  std::lock_guard<std::mutex> lk(p->mu);
  CU(cudaSetDevice(p->device)); CU(cudaDeviceSynchronize());
  if (cycles16) CU(cudaMemcpy(cycles16, p->phase_cycles, 16 * sizeof(unsigned long long), cudaMemcpyDeviceToHost));
  if (reset) CU(cudaMemset(p->phase_cycles, 0, 16 * sizeof(unsigned long long)));
#ifdef FG_PHASE_PROF
  return 1;
#else
  return FG_OK;
#endif
}

static void fill_stats(const HostPlan& H, fg_plan_stats* s) {
  std::memset(s, 0, sizeof(*s));
  s->n_loops = H.g.n; s->M = H.M; s->n_subgraphs = (int)H.subs.size(); s->n_forests = (int)H.forests.size(); s->n_terms = (int)H.terms.size();
  s->n_geoms = (int)H.geoms.size(); s->n_nums = (int)H.nums.size(); s->n_nodes = (int)H.nodes.size();
  s->n_records = H.n_records; s->n_coefs = H.n_coefs; s->n_coefs_nonzero = H.n_nonzero;
  s->stream_bytes = (int64_t)H.d_chunks.size();
  s->flops_per_sample = H.algo_flops; s->exec_flops_per_sample = H.exec_flops; s->plan_seconds = H.plan_seconds;
}
static int dump_structure(const HostPlan& H, int32_t* subs, int32_t* terms, int32_t cap) {
  if (subs) for (size_t k = 0; k < H.subs.size(); ++k) { subs[4 * k] = H.subs[k].a; subs[4 * k + 1] = H.subs[k].b; subs[4 * k + 2] = H.subs[k].type; subs[4 * k + 3] = H.subs[k].chain; }
  int w = 0;
  if (terms) for (auto& t : H.terms) {
    if (w + 3 + 2 * (int)t.members.size() > cap) return fail(FG_E_LIMIT, "terms buffer too small");
    terms[w++] = t.sign; terms[w++] = t.gprime; terms[w++] = (int)t.members.size();
    for (size_t k = 0; k < t.members.size(); ++k) { terms[w++] = t.members[k]; terms[w++] = t.ops[k]; }
  }
  return w;
}

int fg_host_plan(const fg_graph* g, const fg_plan_opts* opts, fg_plan_stats* stats, int32_t* subs, int32_t subs_cap, int32_t* terms, int32_t terms_cap, double* deg, double* Z1) {
  if (!g) return fail(FG_E_ARG, "graph is NULL");
  fg_plan_opts o; if (opts) o = *opts; else fg_plan_opts_default(&o);
  if (o.deg_rule != 0) return fail(FG_E_OPTS, "deg_rule: only rule 0 is available (the paper's Deg algorithm is in its Refs. [42], [32], PAPER.md:250)");
  PlanOpts po; for (int k = 0; k < 4; ++k) po.C[k] = o.C[k]; po.D = o.D; po.merge = o.merge_ext_lines ? 1 : 0;
  po.structure_only = o.structure_only != 0;
  int M = 3 * g->g.n - (po.merge ? 1 : 0);
  if (o.deg_table) po.deg_override.assign(o.deg_table, o.deg_table + ((size_t)1 << M));
  HostPlan H; std::string msg;
  int rc = build_plan(g->g, po, H, msg);
  if (rc != FG_OK) return fail(rc, msg);
  if (stats) fill_stats(H, stats);
  if (subs && (int)H.subs.size() > subs_cap) return fail(FG_E_LIMIT, "subs buffer too small");
  if (deg) std::memcpy(deg, H.deg.data(), H.deg.size() * sizeof(double));
  if (Z1) std::memcpy(Z1, H.Z1.data(), H.Z1.size() * sizeof(double));
  return dump_structure(H, subs, terms, terms_cap);
}

int fg_plan_info(const fg_plan* p, fg_plan_stats* s) {
  if (!p || !s) return fail(FG_E_ARG, "NULL argument");
  fill_stats(p->H, s); s->table_bytes = p->table_bytes; s->wave_samples = (int64_t)p->wave_nb * FG_ST_SAMPLES;
  return FG_OK;
}

int fg_plan_structure(const fg_plan* p, int32_t* subs, int32_t* terms, int32_t cap) {
  if (!p) return fail(FG_E_ARG, "NULL plan");
  return dump_structure(p->H, subs, terms, cap);
}

int fg_host_dirac_table(const fg_graph* g, int32_t a, int32_t b, const int32_t* kids, int32_t n_kids, int32_t op, int32_t comp,
                        const int32_t* pairs, int32_t n_pairs, int32_t qslot, double* table, int32_t table_cap, int32_t* gaps, int32_t* n_gaps) {
  if (!g || !table || !gaps || !n_gaps || (n_kids && !kids) || (n_pairs && !pairs)) return fail(FG_E_ARG, "NULL argument");
  std::vector<std::array<int, 2>> kv, pv;
  for (int k = 0; k < n_kids; ++k) kv.push_back({kids[2 * k], kids[2 * k + 1]});
  for (int k = 0; k < n_pairs; ++k) pv.push_back({pairs[2 * k], pairs[2 * k + 1]});
  std::vector<double> tab; std::vector<int> gp; std::string msg;
  int rc = dirac_table(g->g, a, b, kv, op, comp, pv, qslot, tab, gp, msg);
  if (rc < 0) return fail(rc, msg);
  if ((int)tab.size() > table_cap) return fail(FG_E_LIMIT, "table buffer too small");
  std::memcpy(table, tab.data(), tab.size() * sizeof(double));
  for (size_t k = 0; k < gp.size(); ++k) gaps[k] = gp[k];
  *n_gaps = (int)gp.size();
  return rc;
}

int fg_plan_tables(const fg_plan* p, double* deg, double* Z1) {
  if (!p) return fail(FG_E_ARG, "NULL plan");
  if (deg) std::memcpy(deg, p->H.deg.data(), p->H.deg.size() * sizeof(double));
  if (Z1) std::memcpy(Z1, p->H.Z1.data(), p->H.Z1.size() * sizeof(double));
  return FG_OK;
}

// one slab: double pass, double-double pass over its queue, fold partials
static int run_slab(fg_plan* p, uint64_t first, uint64_t n, uint64_t seed, cudaStream_t st, const double* zin, int mode,
                    double* dI, double* dId, double* dY, double* dErr, uint8_t* dFl, bool finalize, fg_result* out_dev) {
  RunArgs A; std::memset(&A, 0, sizeof(A));
  A.first = first; A.n = n; A.seed = seed; A.zin = zin; A.outI = dI; A.outId = dId; A.outY = dY; A.outErr = dErr; A.outFlags = dFl;
  A.scratch = p->scratch; A.phase_cycles = p->phase_cycles;
  const int nparts = p->grid_d + p->grid_q + p->grid_qd;
  CU(cudaMemsetAsync(p->partials, 0, (size_t)nparts * 8 * sizeof(double), st));
  const uint32_t nwords = (uint32_t)((n + 31) / 32);
  CU(cudaMemsetAsync(p->flag_count, 0, sizeof(unsigned long long), st));
  CU(cudaMemsetAsync(p->flag_count2, 0, sizeof(unsigned long long), st));
  CU(cudaMemsetAsync(p->flag_bits, 0, (size_t)nwords * 4, st));
  CU(cudaMemsetAsync(p->flag_bits2, 0, (size_t)nwords * 4, st));
  cudaEvent_t ev[4] = {nullptr, nullptr, nullptr, nullptr};
  if (p->profile) {
    for (int k = 0; k < 4; ++k) { if (!p->evfree.empty()) { ev[k] = p->evfree.back(); p->evfree.pop_back(); } else CU(cudaEventCreate(&ev[k])); p->evpool.push_back(ev[k]); }
    CU(cudaEventRecord(ev[0], st));
  }
  if (mode <= 1) {          // first rung: double precision; ill-conditioned samples go to the queue of the double-double rung
    A.flag_bits = p->flag_bits; A.do_flag = (mode == 0); A.partials = p->partials;
    A.gV = p->gV; A.gUW = p->gUW; A.gMisc = p->gMisc;
    const uint64_t nbatch = (n + FG_ST_SAMPLES - 1) / FG_ST_SAMPLES;
    for (uint64_t b0 = 0; b0 < nbatch; b0 += (uint64_t)p->wave_nb) {      // waves: geometry of a wave, then its record streams
      A.ord0 = b0 * FG_ST_SAMPLES; A.nb = (int)std::min<uint64_t>((uint64_t)p->wave_nb, nbatch - b0);
      fg_geom_kernel<<<A.nb, FG_ST_SAMPLES, 0, st>>>(p->D, A);
      CU(cudaGetLastError()); ++p->launches;
      fg_stream_kernel<<<std::min(p->grid_d, A.nb), FG_ST_THREADS, p->smem_d, st>>>(p->D, A);
      CU(cudaGetLastError()); ++p->launches;
    }
  }
  if (mode == 0) { fg_compact_kernel<<<1, 1024, 0, st>>>(p->flag_bits, nwords, p->flag_list, p->flag_count); CU(cudaGetLastError()); ++p->launches; }
  if (p->profile) CU(cudaEventRecord(ev[1], st));
  RunArgs B = A; B.phase_cycles = nullptr; B.ord0 = 0; B.nb = 0; B.outId = nullptr;
  if (mode == 0 || mode == 2) {     // second rung: double-double over the queue (mode 2: over every point); its own queue feeds the third
    B.partials = p->partials + (size_t)p->grid_d * 8;
    B.idlist = mode == 0 ? p->flag_list : nullptr; B.idcount = mode == 0 ? p->flag_count : nullptr;
    B.do_flag = 1; B.flag_bits = p->flag_bits2;
    if (mode == 0) B.outErr = nullptr;
    fg_eval_kernel<dd, S_Q, NT_Q><<<p->grid_q, p->nt_q, p->smem_q, st>>>(p->D, B);
    CU(cudaGetLastError()); ++p->launches;
    fg_compact_kernel<<<1, 1024, 0, st>>>(p->flag_bits2, nwords, p->flag_list2, p->flag_count2); CU(cudaGetLastError()); ++p->launches;
  }
  if (mode == 0 || mode == 2 || mode == 3) {     // third rung: quad-double; what it cannot resolve contributes 0
    B.partials = p->partials + (size_t)(p->grid_d + p->grid_q) * 8;
    B.idlist = mode == 3 ? nullptr : p->flag_list2; B.idcount = mode == 3 ? nullptr : p->flag_count2;
    B.do_flag = 0; B.flag_bits = nullptr;
    B.outErr = mode == 3 ? A.outErr : nullptr;
    fg_eval_kernel<qd, 1, NT_QD><<<p->grid_qd, p->nt_qd, p->smem_qd, st>>>(p->D, B);
    CU(cudaGetLastError()); ++p->launches;
  }
  if (p->profile) CU(cudaEventRecord(ev[2], st));
  fg_reduce_kernel<<<1, 32, 0, st>>>(p->partials, nparts, p->accum, (unsigned long long)n, finalize ? 1 : 0, out_dev);
  CU(cudaGetLastError()); ++p->launches;
  if (p->profile) CU(cudaEventRecord(ev[3], st));
  return FG_OK;
}

static int integrate_locked(fg_plan* p, uint64_t first, uint64_t n, uint64_t seed, void* stream, void* out_dev) {
  if (n == 0) return fail(FG_E_ARG, "n_samples must be > 0");
  cudaStream_t st = (cudaStream_t)stream;
  CU(cudaSetDevice(p->device));
  CU(cudaMemsetAsync(p->accum, 0, sizeof(Accum), st));
  for (uint64_t done = 0; done < n; done += SLAB) {
    uint64_t m = std::min<uint64_t>(SLAB, n - done);
    int rc = run_slab(p, first + done, m, seed, st, nullptr, 0, nullptr, nullptr, nullptr, nullptr, nullptr, done + m >= n, (fg_result*)out_dev);
    if (rc != FG_OK) return rc;
  }
  return FG_OK;
}

int fg_integrate_async(const fg_plan* cp, uint64_t first, uint64_t n, uint64_t seed, void* stream, void* out_dev) {
  fg_plan* p = const_cast<fg_plan*>(cp);
  if (!p || !out_dev) return fail(FG_E_ARG, "NULL argument");
  std::lock_guard<std::mutex> lk(p->mu);      // the launches of one call are enqueued atomically; see fg.h for stream rules
  return integrate_locked(p, first, n, seed, stream, out_dev);
}

int fg_integrate_range(const fg_plan* cp, uint64_t first, uint64_t n, uint64_t seed, void* stream, fg_result* out) {
  fg_plan* p = const_cast<fg_plan*>(cp);
  if (!p || !out) return fail(FG_E_ARG, "NULL argument");
  std::lock_guard<std::mutex> lk(p->mu);
  int rc = integrate_locked(p, first, n, seed, stream, p->result_dev);
  if (rc != FG_OK) return rc;
  CU(cudaMemcpyAsync(out, p->result_dev, sizeof(fg_result), cudaMemcpyDeviceToHost, (cudaStream_t)stream));
  CU(cudaStreamSynchronize((cudaStream_t)stream));
  return FG_OK;
}
int fg_integrate(const fg_plan* p, uint64_t n, uint64_t seed, void* stream, fg_result* out) { return fg_integrate_range(p, 0, n, seed, stream, out); }

int fg_result_merge(const fg_result* a, const fg_result* b, fg_result* out) {
  if (!a || !b || !out) return fail(FG_E_ARG, "NULL argument");
  fg_result r; std::memset(&r, 0, sizeof(r));
  dd sy = dd(a->sum_y[0], a->sum_y[1]) + dd(b->sum_y[0], b->sum_y[1]);
  dd s2 = dd(a->sum_y2[0], a->sum_y2[1]) + dd(b->sum_y2[0], b->sum_y2[1]);
  r.n_samples = a->n_samples + b->n_samples; r.n_flagged = a->n_flagged + b->n_flagged; r.n_rejected = a->n_rejected + b->n_rejected;
  r.n_pdf_big_exp = a->n_pdf_big_exp + b->n_pdf_big_exp;
  r.sum_y[0] = sy.hi; r.sum_y[1] = sy.lo; r.sum_y2[0] = s2.hi; r.sum_y2[1] = s2.lo;
  double N = (double)r.n_samples;
  if (N > 0) { r.mean = to_double(sy) / N; r.variance = to_double(s2 / dd(N * N) - sy * sy / dd(N * N * N)); }
  *out = r; return FG_OK;
}

// ---- debug / parity surface -----------------------------------------------------------------------------------
struct DevBuf {
  void* d = nullptr; size_t bytes = 0;
  ~DevBuf() { if (d) cudaFree(d); }
  cudaError_t alloc(size_t b) { bytes = b; return cudaMalloc(&d, std::max<size_t>(b, 16)); }
};
#define CUB(x) do { cudaError_t e_ = (x); if (e_ != cudaSuccess) return fail(FG_E_CUDA, std::string(#x) + ": " + cudaGetErrorString(e_)); } while (0)

int fg_sample_dump(const fg_plan* cp, uint64_t first, uint64_t n, uint64_t seed, void* stream, uint32_t* words, int32_t* comp,
                   uint8_t* order, double* z, double* mant, int32_t* ex, uint8_t* bad) {
  fg_plan* p = const_cast<fg_plan*>(cp);
  if (!p) return fail(FG_E_ARG, "NULL plan");
  if (n == 0) return FG_OK;
  cudaStream_t st = (cudaStream_t)stream; CU(cudaSetDevice(p->device));
  const int M = p->D.M;
  DevBuf bw, bc, bo, bz, bm, be, bb;
  if (words) CUB(bw.alloc(n * M * 4 * sizeof(uint32_t))); if (comp) CUB(bc.alloc(n * sizeof(int32_t))); if (order) CUB(bo.alloc(n * M));
  if (z) CUB(bz.alloc(n * M * sizeof(double))); if (mant) CUB(bm.alloc(n * sizeof(double))); if (ex) CUB(be.alloc(n * sizeof(int32_t))); if (bad) CUB(bb.alloc(n));
  fg_sample_dump_kernel<<<(unsigned)((n + 127) / 128), 128, 0, st>>>(p->D, first, n, seed, (uint32_t*)bw.d, (int32_t*)bc.d, (uint8_t*)bo.d, (double*)bz.d, (double*)bm.d, (int32_t*)be.d, (uint8_t*)bb.d);
  CU(cudaGetLastError());
  auto back = [&](void* h, DevBuf& b) { return h ? cudaMemcpyAsync(h, b.d, b.bytes, cudaMemcpyDeviceToHost, st) : cudaSuccess; };
  CU(back(words, bw)); CU(back(comp, bc)); CU(back(order, bo)); CU(back(z, bz)); CU(back(mant, bm)); CU(back(ex, be)); CU(back(bad, bb));
  CU(cudaStreamSynchronize(st));
  return FG_OK;
}

static int eval_common(fg_plan* p, const double* z_host, uint64_t first, uint64_t n, uint64_t seed, int mode, cudaStream_t st,
                       double* I, double* Id, double* Y, double* err, uint8_t* flags) {
  if (n == 0) return FG_OK;
  if (n > SLAB) return fail(FG_E_ARG, "at most 2^24 points per call");
  std::lock_guard<std::mutex> lk(p->mu);
  CU(cudaSetDevice(p->device));
  const int M = p->D.M;
  DevBuf bz, bI, bId, bY, bE, bF;
  if (z_host) { CUB(bz.alloc(n * M * sizeof(double))); CU(cudaMemcpyAsync(bz.d, z_host, bz.bytes, cudaMemcpyHostToDevice, st)); }
  CUB(bI.alloc(n * sizeof(double))); CUB(bId.alloc(n * sizeof(double))); CUB(bY.alloc(n * sizeof(double))); CUB(bE.alloc(n * sizeof(double))); CUB(bF.alloc(n));
  CU(cudaMemsetAsync(bF.d, 0, n, st)); CU(cudaMemsetAsync(bE.d, 0, n * sizeof(double), st)); CU(cudaMemsetAsync(bId.d, 0, n * sizeof(double), st));
  CU(cudaMemsetAsync(p->accum, 0, sizeof(Accum), st));
  int rc = run_slab(p, first, n, seed, st, (const double*)bz.d, mode, (double*)bI.d, (double*)bId.d, (double*)bY.d, (double*)bE.d, (uint8_t*)bF.d, true, p->result_dev);
  if (rc != FG_OK) return rc;
  auto back = [&](void* h, DevBuf& b) { return h ? cudaMemcpyAsync(h, b.d, b.bytes, cudaMemcpyDeviceToHost, st) : cudaSuccess; };
  CU(back(I, bI)); CU(back(Id, bId)); CU(back(Y, bY)); CU(back(err, bE)); CU(back(flags, bF));
  CU(cudaStreamSynchronize(st));
  return FG_OK;
}

int fg_eval_points(const fg_plan* cp, const double* z, uint64_t n, int32_t mode, void* stream, double* I, double* I_double, double* err, uint8_t* flags) {
  if (!cp || (!z && n)) return fail(FG_E_ARG, "NULL argument");
  if (mode < 0 || mode > 3) return fail(FG_E_ARG, "mode must be 0, 1, 2 or 3");
  return eval_common(const_cast<fg_plan*>(cp), z, 0, n, 0, mode, (cudaStream_t)stream, I, I_double, nullptr, err, flags);
}

int fg_sample_eval_dump(const fg_plan* cp, uint64_t first, uint64_t n, uint64_t seed, void* stream, double* I, double* y, uint8_t* flags) {
  if (!cp) return fail(FG_E_ARG, "NULL plan");
  return eval_common(const_cast<fg_plan*>(cp), nullptr, first, n, seed, 0, (cudaStream_t)stream, I, nullptr, y, nullptr, flags);
}

// ---- no-allocation entry point -----------------------------------------------------------------------------------------
// For callers that cannot call cudaMalloc (code under CUDA graph capture, tight serving loops, harnesses that forbid it):
// the double-double evaluation of given points with the per-block scratch of fg_eval_kernel<dd> in a file-scope device
// array instead of the plan's cudaMalloc'ed scratch.  Every GPU that loads the library holds the array until exit.
#define FG_NOALLOC_SCRATCH_BYTES (32u << 20)        // 32 MiB
#define FG_NOALLOC_MAX_POINTS (1u << 20)
static __device__ __align__(256) unsigned char fg_noalloc_scratch[FG_NOALLOC_SCRATCH_BYTES];
// In host code `fg_noalloc_scratch` is a host-side stand-in, not a device address: the address the kernel gets comes from
// cudaGetSymbolAddress, once per device, with that device current.
static std::mutex g_noalloc_mu;
static void* g_noalloc_ptr[64] = {nullptr};

static int noalloc_setup_locked(int device) {
  if (device < 0 || device >= 64) return fail(FG_E_ARG, "device out of range");
  if (g_noalloc_ptr[device]) return FG_OK;
  CU(cudaSetDevice(device));
  void* ptr = nullptr;
  cudaError_t e = cudaGetSymbolAddress((void**)&ptr, fg_noalloc_scratch);
  if (e != cudaSuccess || !ptr) return fail(FG_E_CUDA, std::string("cudaGetSymbolAddress(fg_noalloc_scratch): ") + cudaGetErrorString(e));
  g_noalloc_ptr[device] = ptr;
  return FG_OK;
}

int fg_noalloc_setup(int32_t device) {
  int ndev = 0; if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) return fail(FG_E_CUDA, "no CUDA device");
  if (device < 0 || device >= ndev) return fail(FG_E_ARG, "device out of range");
  std::lock_guard<std::mutex> lk(g_noalloc_mu);
  return noalloc_setup_locked(device);
}

int fg_noalloc_limits(uint64_t* scratch_bytes, uint64_t* max_points) {
  if (scratch_bytes) *scratch_bytes = FG_NOALLOC_SCRATCH_BYTES;
  if (max_points) *max_points = FG_NOALLOC_MAX_POINTS;
  return FG_OK;
}

int fg_eval_points_dd_noalloc(const fg_plan* cp, const double* z_dev, uint64_t n, void* stream, double* I_dev, double* err_dev, uint8_t* flags_dev) {
  fg_plan* p = const_cast<fg_plan*>(cp);
  if (!p || !z_dev || !I_dev || !flags_dev) return fail(FG_E_ARG, "NULL argument");
  if (n == 0) return FG_OK;
  if (n > FG_NOALLOC_MAX_POINTS) return fail(FG_E_LIMIT, "fg_eval_points_dd_noalloc: at most 2^20 points per call");
  const size_t per_block = (size_t)p->D.scratch_slots * (size_t)p->nt_q * S_Q * sizeof(dd);
  if (per_block > FG_NOALLOC_SCRATCH_BYTES)
    return fail(FG_E_LIMIT, "fg_eval_points_dd_noalloc: the per-block scratch of this plan (" + std::to_string(per_block) + " bytes) exceeds the static array (" + std::to_string((size_t)FG_NOALLOC_SCRATCH_BYTES) + " bytes)");
  { std::lock_guard<std::mutex> lk(g_noalloc_mu); int rc = noalloc_setup_locked(p->device); if (rc != FG_OK) return rc; }
  std::lock_guard<std::mutex> lk(p->mu);
  cudaStream_t st = (cudaStream_t)stream;
  CU(cudaSetDevice(p->device));
  const int grid = (int)std::min<size_t>((size_t)p->grid_q, FG_NOALLOC_SCRATCH_BYTES / per_block);
  RunArgs B; std::memset(&B, 0, sizeof(B));
  B.n = n; B.zin = z_dev; B.outI = I_dev; B.outErr = err_dev; B.outFlags = flags_dev;
  B.scratch = g_noalloc_ptr[p->device];
  B.partials = p->partials + (size_t)p->grid_d * 8;           // plan-owned (allocated by fg_plan_create); the sums are not returned
  B.do_flag = 0;                                               // last rung of this call: unresolved points get flag bit 2
  // the array keeps the last call's contents: the kernel writes every scratch slot before it reads it, but the part this
  // launch uses is cleared all the same, and so are the flags (the kernel ORs into them) and the partial sums it adds to
  CU(cudaMemsetAsync(B.scratch, 0, (size_t)grid * per_block, st));
  CU(cudaMemsetAsync(flags_dev, 0, n, st));
  CU(cudaMemsetAsync(B.partials, 0, (size_t)p->grid_q * 8 * sizeof(double), st));
  fg_eval_kernel<dd, S_Q, NT_Q><<<grid, p->nt_q, p->smem_q, st>>>(p->D, B);
  CU(cudaGetLastError()); ++p->launches;
  return FG_OK;
}

int fg_dfma_peak(int32_t device, int32_t iters, void* stream, double* tflops, double* ms_out) {
  if (!tflops || iters <= 0) return fail(FG_E_ARG, "bad argument");
  int ndev = 0; if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) return fail(FG_E_CUDA, "no CUDA device");
  CU(cudaSetDevice(device));
  cudaDeviceProp prop; CU(cudaGetDeviceProperties(&prop, device));
  cudaStream_t st = (cudaStream_t)stream;
  const int threads = 256, blocks = prop.multiProcessorCount * 8;
  DevBuf out; CUB(out.alloc((size_t)threads * blocks * sizeof(double)));
  cudaEvent_t e0, e1; CU(cudaEventCreate(&e0)); CU(cudaEventCreate(&e1));
  fg_dfma_kernel<<<blocks, threads, 0, st>>>((double*)out.d, iters / 8 + 1, 0.999999, 1e-7);   // warm-up
  CU(cudaEventRecord(e0, st));
  fg_dfma_kernel<<<blocks, threads, 0, st>>>((double*)out.d, iters, 0.999999, 1e-7);
  CU(cudaEventRecord(e1, st)); CU(cudaEventSynchronize(e1));
  float ms = 0; CU(cudaEventElapsedTime(&ms, e0, e1));
  cudaEventDestroy(e0); cudaEventDestroy(e1);
  double flops = 2.0 * 8.0 * (double)iters * threads * blocks;
  *tflops = flops / (ms * 1e-3) / 1e12; if (ms_out) *ms_out = ms;
  return FG_OK;
}

int fg_dmma_peak(int32_t device, int32_t iters, void* stream, double* tflops, double* ms_out) {
  if (!tflops || iters <= 0) return fail(FG_E_ARG, "bad argument");
  int ndev = 0; if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) return fail(FG_E_CUDA, "no CUDA device");
  CU(cudaSetDevice(device));
  cudaDeviceProp prop; CU(cudaGetDeviceProperties(&prop, device));
  cudaStream_t st = (cudaStream_t)stream;
  const int threads = 256, blocks = prop.multiProcessorCount * 8;
  DevBuf out; CUB(out.alloc((size_t)threads * blocks * sizeof(double)));
  cudaEvent_t e0, e1; CU(cudaEventCreate(&e0)); CU(cudaEventCreate(&e1));
  fg_dmma_kernel<<<blocks, threads, 0, st>>>((double*)out.d, iters / 8 + 1, 1e-3, 1.0);   // warm-up
  CU(cudaEventRecord(e0, st));
  fg_dmma_kernel<<<blocks, threads, 0, st>>>((double*)out.d, iters, 1e-3, 1.0);
  CU(cudaEventRecord(e1, st)); CU(cudaEventSynchronize(e1));
  float ms = 0; CU(cudaEventElapsedTime(&ms, e0, e1));
  cudaEventDestroy(e0); cudaEventDestroy(e1);
  const double flops = 2.0 * 8 * 8 * 4 * 8.0 * (double)iters * ((double)threads * blocks / 32.0);
  *tflops = flops / (ms * 1e-3) / 1e12; if (ms_out) *ms_out = ms;
  return FG_OK;
}

}  // extern "C"
