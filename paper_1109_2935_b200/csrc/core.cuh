// core.cuh -- packed field records, precision traits, SU(3) link reconstruction.
//
// Data layout in HBM: every field is an even-odd checkerboarded
// structure of arrays.  A record of N reals of storage type T (N*sizeof(T) bytes per site)
// is split into 16-byte chunks (then one 8- and/or one 4-byte chunk); chunk k of all sites is
// one contiguous plane, so a warp reading chunk k of 32 consecutive sites issues one fully
// coalesced 512-byte (int4) request.  (PAPER.md:164, :180-186 and Figs. 2,3 describe the
// same idea for Fermi with float2/float4 textures; the chunking here is sized for 128-bit
// loads on sm_100a.)
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace lq {

// Geometry of one launch: a batch of `nb` independent 4-d boxes of extents X (one box = the
// whole lattice for the global operator; one box = one Schwarz block for the Dirichlet
// operator).  bc[mu]: +1 periodic, -1 antiperiodic, 0 open (hop dropped).
struct Geom {
  int X[4];
  int Xh;          // X[0]/2
  signed char bc[4];   // +1 periodic, -1 antiperiodic, 0 open (Dirichlet) per direction
  int vh;          // sites of one parity in one box
  int nb;          // boxes in the batch
  long long ns;    // nb*vh = plane stride of every packed field
  // ceil(2^32 / d) for d = Xh, X[1], X[2]: n / d = umulhi(n, m) exactly for n d < 2^32 (checked where a Geom is made);
  // the three run-time divisions of the site index were ~50 instructions and 9 XU-pipe operations per thread
  unsigned mXh, mY, mZ;
};
static_assert(sizeof(Geom) == 56, "Geom is part of DslashArgs, which must stay 128 bytes (dslash.cuh)");

struct PrecD { typedef double store_t; typedef double real; static constexpr bool HALF = false; static constexpr int ID = 0; };
struct PrecS { typedef float  store_t; typedef float  real; static constexpr bool HALF = false; static constexpr int ID = 1; };
struct PrecH { typedef short  store_t; typedef float  real; static constexpr bool HALF = true;  static constexpr int ID = 2; };

#define LQ_DEV __device__ __forceinline__
#ifndef LQ_GAUGE_STREAM
#define LQ_GAUGE_STREAM 1
#endif

// Debug build (LQ_EXTRA_FLAGS=-DLQ_BOUNDS_CHECK sh build.sh): every record index of every packed
// field access is checked against the field's record count and the kernel traps on a violation
// (compute-sanitizer is not available on the GPU pool this was developed on).
#ifdef LQ_BOUNDS_CHECK
#define LQ_CHECK_INDEX(i, ns) do { if ((unsigned long long)(i) >= (unsigned long long)(ns)) __trap(); } while (0)
#else
#define LQ_CHECK_INDEX(i, ns) do { } while (0)
#endif

template <typename V> LQ_DEV V ld_nc(const V* p) { return __ldg(p); }
// streaming variants for data with no reuse (gauge links): do not allocate in L1
LQ_DEV int4 ld_stream(const int4* p) {
  int4 v;
  asm volatile("ld.global.nc.L1::no_allocate.v4.s32 {%0,%1,%2,%3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "l"(p));
  return v;
}
LQ_DEV int2 ld_stream(const int2* p) {
  int2 v;
  asm volatile("ld.global.nc.L1::no_allocate.v2.s32 {%0,%1}, [%2];" : "=r"(v.x), "=r"(v.y) : "l"(p));
  return v;
}
LQ_DEV unsigned smem_addr(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
LQ_DEV int4 ld_shared(const int4* p) {
  int4 v;
  asm volatile("ld.shared.v4.s32 {%0,%1,%2,%3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(smem_addr(p)) : "memory");
  return v;
}
LQ_DEV int2 ld_shared(const int2* p) {
  int2 v;
  asm volatile("ld.shared.v2.s32 {%0,%1}, [%2];" : "=r"(v.x), "=r"(v.y) : "r"(smem_addr(p)) : "memory");
  return v;
}
LQ_DEV int ld_shared(const int* p) {
  int v;
  asm volatile("ld.shared.s32 %0, [%1];" : "=r"(v) : "r"(smem_addr(p)) : "memory");
  return v;
}
// asynchronous global -> shared copies (LDGSTS): the bytes in flight occupy no registers
template <int BYTES> LQ_DEV void cp_async(void* smem_dst, const void* gsrc) {
  if constexpr (BYTES == 16)
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(smem_addr(smem_dst)), "l"(gsrc) : "memory");
  else if constexpr (BYTES == 8)
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(smem_addr(smem_dst)), "l"(gsrc) : "memory");
  else
    asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(smem_addr(smem_dst)), "l"(gsrc) : "memory");
}
LQ_DEV void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N> LQ_DEV void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

LQ_DEV int ld_stream(const int* p) {
  int v;
  asm volatile("ld.global.nc.L1::no_allocate.s32 %0, [%1];" : "=r"(v) : "l"(p));
  return v;
}

// ---------------------------------------------------------------- packed records
template <typename T, int N>
struct Rec {
  static constexpr int BYTES = N * (int)sizeof(T);
  static constexpr int N16 = BYTES / 16;
  static constexpr int N8 = (BYTES % 16) / 8;
  static constexpr int N4 = (BYTES % 8) / 4;
  static constexpr int E16 = 16 / (int)sizeof(T), E8 = 8 / (int)sizeof(T), E4 = 4 / (int)sizeof(T);
  static_assert(BYTES % 4 == 0, "record must be a multiple of 4 bytes");

  // MODE 0: read-only global (ld.global.nc), 1: streaming global (no L1 allocation),
  // 2: shared memory staging buffer laid out like a packed field with ns = CTA size, i = thread
  template <int MODE = 0>
  LQ_DEV static void load(T* __restrict__ v, const char* __restrict__ base, long long ns, long long i) {
    LQ_CHECK_INDEX(i, ns);
#pragma unroll
    for (int k = 0; k < N16; ++k) {
      const int4* p = reinterpret_cast<const int4*>(base + 16ll * k * ns) + i;
      int4 t = MODE == 2 ? ld_shared(p) : MODE == 1 ? ld_stream(p) : ld_nc(p);
      *reinterpret_cast<int4*>(v + k * E16) = t;
    }
    if (N8) {
      const int2* p = reinterpret_cast<const int2*>(base + 16ll * N16 * ns) + i;
      int2 t = MODE == 2 ? ld_shared(p) : MODE == 1 ? ld_stream(p) : ld_nc(p);
      *reinterpret_cast<int2*>(v + N16 * E16) = t;
    }
    if (N4) {
      const int* p = reinterpret_cast<const int*>(base + (16ll * N16 + 8ll * N8) * ns) + i;
      int t = MODE == 2 ? ld_shared(p) : MODE == 1 ? ld_stream(p) : ld_nc(p);
      *reinterpret_cast<int*>(v + N16 * E16 + N8 * E8) = t;
    }
  }
  // record i of the global field -> record `tid` of a staging buffer of `nt` records
  LQ_DEV static void stage(char* __restrict__ sbase, int nt, int tid, const char* __restrict__ base, long long ns, long long i) {
    LQ_CHECK_INDEX(i, ns);
    LQ_CHECK_INDEX(tid, nt);
#pragma unroll
    for (int k = 0; k < N16; ++k)
      cp_async<16>(sbase + 16 * k * nt + 16 * tid, reinterpret_cast<const int4*>(base + 16ll * k * ns) + i);
    if (N8) cp_async<8>(sbase + 16 * N16 * nt + 8 * tid, reinterpret_cast<const int2*>(base + 16ll * N16 * ns) + i);
    if (N4) cp_async<4>(sbase + (16 * N16 + 8 * N8) * nt + 4 * tid, reinterpret_cast<const int*>(base + (16ll * N16 + 8ll * N8) * ns) + i);
  }
  LQ_DEV static void store(const T* __restrict__ v, char* __restrict__ base, long long ns, long long i) {
    LQ_CHECK_INDEX(i, ns);
#pragma unroll
    for (int k = 0; k < N16; ++k)
      reinterpret_cast<int4*>(base + 16ll * k * ns)[i] = *reinterpret_cast<const int4*>(v + k * E16);
    if (N8) reinterpret_cast<int2*>(base + 16ll * N16 * ns)[i] = *reinterpret_cast<const int2*>(v + N16 * E16);
    if (N4) reinterpret_cast<int*>(base + (16ll * N16 + 8ll * N8) * ns)[i] = *reinterpret_cast<const int*>(v + N16 * E16 + N8 * E8);
  }
};

// bytes per site of a packed field of N reals (+ one fp32 norm per site in half precision)
template <class P> __host__ __device__ constexpr int site_bytes(int n, bool with_norm) {
  return n * (int)sizeof(typename P::store_t) + ((P::HALF && with_norm) ? 4 : 0);
}

#define LQ_FIXED_MAX 32767.0f
#define LQ_FIXED_INV (1.0f / 32767.0f)
// 16-bit fixed point is stored in offset binary (u = q + 32768, q in [-32767, 32767]) so that
// decoding is one byte-permute into the mantissa of 2^23 and one FADD, and encoding is one FFMA
// whose result's low 16 bits are u (round-to-nearest-even done by the FP adder); no I2F / F2I.
#define LQ_MAGIC_DEC 8421376.0f      /* 2^23 + 32768 */
#define LQ_MAGIC_ENC 12615680.0f     /* 1.5*2^23 + 32768 */

LQ_DEV float fma_(float a, float b, float c) { return fmaf(a, b, c); }
LQ_DEV double fma_(double a, double b, double c) { return fma(a, b, c); }

// ---------------------------------------------------------------- packed fp32 pairs (FFMA2 / FADD2 / FMUL2, sm_100)
// A complex number (re, im) held in one aligned 64-bit register pair.  The fp32-arithmetic kernels are bound by
// register-file bandwidth, not by the FMA lanes: a scalar FFMA reads three registers and, measured on B200 with
// the SU(3) x half-spinor product of dslash.cuh, sustains 0.62 FFMA/clk/scheduler; the packed form
//   (re, im) += u.re * (h.re, h.im);   (re, im) += u.im * (-h.im, h.re)
// is two FFMA2 whose scalar factor is a broadcast operand (.F32) and whose swapped / half-negated pair is an operand
// modifier (.LO_HI, .NP / .PN) -- ptxas folds f2_make(u, u) and f2_make(-b, a) into those -- and sustains 0.85
// FMA-equivalents/clk (175 -> 128 clk per hop).  Each lane is an IEEE fma, so results are
// bit-identical to the scalar sequence with the same per-component order.
typedef unsigned long long f2;
LQ_DEV f2 f2_make(float lo, float hi) { f2 r; asm("mov.b64 %0, {%1,%2};" : "=l"(r) : "f"(lo), "f"(hi)); return r; }
LQ_DEV f2 f2_bcast(float x) { return f2_make(x, x); }
LQ_DEV void f2_split(f2 v, float& lo, float& hi) { asm("mov.b64 {%0,%1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v)); }
LQ_DEV f2 f2_fma(f2 a, f2 b, f2 c) { f2 d; asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c)); return d; }
LQ_DEV f2 f2_mul(f2 a, f2 b) { f2 d; asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b)); return d; }
LQ_DEV f2 f2_add(f2 a, f2 b) { f2 d; asm("add.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b)); return d; }

// the two 16-bit fields of w as floats holding the signed integers q
LQ_DEV float fixed_lo(unsigned w) { return __uint_as_float(__byte_perm(w, 0x4B000000u, 0x7610)) - LQ_MAGIC_DEC; }
LQ_DEV float fixed_hi(unsigned w) { return __uint_as_float(__byte_perm(w, 0x4B000000u, 0x7632)) - LQ_MAGIC_DEC; }
// both fields of w at once: two PRMT and one FADD2
LQ_DEV void fixed_pair(unsigned w, float& lo, float& hi) {
  const f2 m = f2_make(__uint_as_float(__byte_perm(w, 0x4B000000u, 0x7610)), __uint_as_float(__byte_perm(w, 0x4B000000u, 0x7632)));
  f2_split(f2_add(m, f2_bcast(-LQ_MAGIC_DEC)), lo, hi);
}
// pack rint(a*sc), rint(b*sc) (|.| <= 32767) as two offset-binary 16-bit fields
LQ_DEV unsigned fixed_pack(float a, float b, float sc) {
  float ea, eb;
  f2_split(f2_fma(f2_make(a, b), f2_bcast(sc), f2_bcast(LQ_MAGIC_ENC)), ea, eb);
  return __byte_perm(__float_as_uint(ea), __float_as_uint(eb), 0x5410);
}

// ---------------------------------------------------------------- site vectors with a norm (spinor: 24, clover: 72)
// R9: half = 16-bit fixed point q_i = rint(v_i * 32767 / n), n = max_i |v_i| (fp32) per site; decode v_i = q_i * n/32767.
// load_site_raw returns v and scale with (true value) = scale * v, so that callers can fold
// the scale into an FMA coefficient instead of spending one FMUL per element.
template <class P, int N, int MODE = 0>
LQ_DEV void load_site_raw(typename P::real* __restrict__ v, typename P::real& scale, const char* __restrict__ f, long long ns, long long i) {
  if constexpr (!P::HALF) {
    Rec<typename P::store_t, N>::template load<MODE>(v, f, ns, i);
    scale = 1;
  } else {
    alignas(16) unsigned w[N / 2];
    Rec<unsigned, N / 2>::template load<MODE>(w, f, ns, i);
    const int* np = reinterpret_cast<const int*>(f + (long long)(2 * N) * ns) + i;
    scale = __int_as_float(MODE == 2 ? ld_shared(np) : ld_nc(np)) * LQ_FIXED_INV;
#pragma unroll
    for (int k = 0; k < N / 2; ++k) fixed_pair(w[k], v[2 * k], v[2 * k + 1]);
  }
}

// half precision only: the N stored values as floats m = 2^23 + 32768 + q (no decoding FADD), for consumers that
// combine pairs of them exactly (fixed_project in dslash.cuh); scale as in load_site_raw
template <class P, int N, int MODE = 0>
LQ_DEV void load_site_magic(float* __restrict__ m, float& scale, const char* __restrict__ f, long long ns, long long i) {
  static_assert(P::HALF, "magic-float form exists for the 16-bit fixed-point storage only");
  alignas(16) unsigned w[N / 2];
  Rec<unsigned, N / 2>::template load<MODE>(w, f, ns, i);
  const int* np = reinterpret_cast<const int*>(f + (long long)(2 * N) * ns) + i;
  scale = __int_as_float(MODE == 2 ? ld_shared(np) : ld_nc(np)) * LQ_FIXED_INV;
#pragma unroll
  for (int k = 0; k < N / 2; ++k) {
    m[2 * k] = __uint_as_float(__byte_perm(w[k], 0x4B000000u, 0x7610));
    m[2 * k + 1] = __uint_as_float(__byte_perm(w[k], 0x4B000000u, 0x7632));
  }
}

template <class P, int N>
LQ_DEV void load_site(typename P::real* __restrict__ v, const char* __restrict__ f, long long ns, long long i) {
  typename P::real sc;
  load_site_raw<P, N>(v, sc, f, ns, i);
  if constexpr (P::HALF) {
#pragma unroll
    for (int k = 0; k < N; ++k) v[k] *= sc;
  }
}

template <class P, int N>
LQ_DEV void store_site(const typename P::real* __restrict__ v, char* __restrict__ f, long long ns, long long i) {
  if constexpr (!P::HALF) {
    Rec<typename P::store_t, N>::store(v, f, ns, i);
  } else {
    float m = 0.f;
#pragma unroll
    for (int k = 0; k < N; ++k) m = fmaxf(m, fabsf(v[k]));
    const float sc = (m > 0.f) ? (LQ_FIXED_MAX / m) : 0.f;
    alignas(16) unsigned w[N / 2];
#pragma unroll
    for (int k = 0; k < N / 2; ++k) w[k] = fixed_pack(v[2 * k], v[2 * k + 1], sc);
    Rec<unsigned, N / 2>::store(w, f, ns, i);
    reinterpret_cast<float*>(f + (long long)(2 * N) * ns)[i] = m;
  }
}

// ---------------------------------------------------------------- complex helpers on (re,im) pairs
template <typename R> struct cx { R re, im; };
template <typename R> LQ_DEV cx<R> cmul(cx<R> a, cx<R> b) { return {a.re * b.re - a.im * b.im, a.re * b.im + a.im * b.re}; }
template <typename R> LQ_DEV cx<R> cmulc(cx<R> a, cx<R> b) { /* conj(a)*b */ return {a.re * b.re + a.im * b.im, a.re * b.im - a.im * b.re}; }
template <typename R> LQ_DEV cx<R> conj_(cx<R> a) { return {a.re, -a.im}; }

LQ_DEV void sincos_(float x, float* s, float* c) { __sincosf(x, s, c); }
LQ_DEV void sincos_(double x, double* s, double* c) { sincos(x, s, c); }
LQ_DEV float rsqrt_(float x) { return rsqrtf(x); }
LQ_DEV double rsqrt_(double x) { return rsqrt(x); }
LQ_DEV float sqrt_(float x) { return sqrtf(x); }
LQ_DEV double sqrt_(double x) { return sqrt(x); }

// ---------------------------------------------------------------- gauge links (PAPER.md:164 (a); R10)
// u[18] = row-major 3x3 complex with (true link) = uscale * u.  RECON 18: as stored.  12: rows
// 0,1 stored, row2 = conj(row0 x row1).  8: a2,a3,b1,arg(a1),arg(c1) stored (the
// parametrisation of ref. [3] of the paper).  In half precision the 16-bit integers are kept
// unscaled (uscale = 1/32767 is folded into the caller's accumulate coefficient).
template <class P, int RECON, int MODE = LQ_GAUGE_STREAM>
LQ_DEV void load_link(typename P::real* __restrict__ u, typename P::real& uscale, const char* __restrict__ g, long long ns, long long i) {
  typedef typename P::real R;
  R v[RECON];
  if constexpr (P::HALF) {
    alignas(16) unsigned w[RECON / 2];
    Rec<unsigned, RECON / 2>::template load<MODE>(w, g, ns, i);
#pragma unroll
    for (int k = 0; k < RECON / 2; ++k) fixed_pair(w[k], v[2 * k], v[2 * k + 1]);
    if constexpr (RECON == 8) {
#pragma unroll
      for (int k = 0; k < 6; ++k) v[k] *= LQ_FIXED_INV;
      v[6] *= 3.14159265358979323846f * LQ_FIXED_INV; v[7] *= 3.14159265358979323846f * LQ_FIXED_INV;
      uscale = 1;
    } else {
      uscale = LQ_FIXED_INV;
    }
  } else {
    Rec<typename P::store_t, RECON>::template load<MODE>(v, g, ns, i);
    uscale = 1;
  }
  if constexpr (RECON == 18) {
#pragma unroll
    for (int k = 0; k < 18; ++k) u[k] = v[k];
  } else if constexpr (RECON == 12 && sizeof(R) == 4) {
#pragma unroll
    for (int k = 0; k < 12; ++k) u[k] = v[k];
    // row2 = conj(row0 x row1), packed: (re, im) of conj(a_j b_k - a_k b_j) in four FFMA2 (a = row 0, b = row 1)
#pragma unroll
    for (int c = 0; c < 3; ++c) {
      const int j = (c + 1) % 3, k = (c + 2) % 3;
      const float ajr = u[2 * j], aji = u[2 * j + 1], akr = u[2 * k], aki = u[2 * k + 1];
      const float bjr = u[6 + 2 * j], bji = u[6 + 2 * j + 1], bkr = u[6 + 2 * k], bki = u[6 + 2 * k + 1];
      f2 t = f2_mul(f2_make(bkr, -bki), f2_bcast(ajr));
      t = f2_fma(f2_make(-bki, -bkr), f2_bcast(aji), t);
      t = f2_fma(f2_make(-bjr, bji), f2_bcast(akr), t);
      t = f2_fma(f2_make(bji, bjr), f2_bcast(aki), t);
      if constexpr (P::HALF) t = f2_mul(t, f2_bcast(LQ_FIXED_INV));
      float re, im;
      f2_split(t, re, im);
      u[12 + 2 * c] = re;
      u[12 + 2 * c + 1] = im;
    }
  } else if constexpr (RECON == 12) {
#pragma unroll
    for (int k = 0; k < 12; ++k) u[k] = v[k];
    // row2 = conj(row0 x row1) (times uscale, so that all three rows carry the same scale)
#pragma unroll
    for (int c = 0; c < 3; ++c) {
      const int j = (c + 1) % 3, k = (c + 2) % 3;
      R re = u[2 * j] * u[6 + 2 * k];
      re = fma_(-u[2 * j + 1], u[6 + 2 * k + 1], re);
      re = fma_(-u[2 * k], u[6 + 2 * j], re);
      re = fma_(u[2 * k + 1], u[6 + 2 * j + 1], re);
      R im = u[2 * k] * u[6 + 2 * j + 1];
      im = fma_(u[2 * k + 1], u[6 + 2 * j], im);
      im = fma_(-u[2 * j], u[6 + 2 * k + 1], im);
      im = fma_(-u[2 * j + 1], u[6 + 2 * k], im);
      if constexpr (P::HALF) { re *= LQ_FIXED_INV; im *= LQ_FIXED_INV; }
      u[12 + 2 * c] = re;
      u[12 + 2 * c + 1] = im;
    }
  } else {
    const cx<R> a2 = {v[0], v[1]}, a3 = {v[2], v[3]}, b1 = {v[4], v[5]};
    const R N = a2.re * a2.re + a2.im * a2.im + a3.re * a3.re + a3.im * a3.im;
    R s1, c1, s2, c2;
    sincos_(v[6], &s1, &c1);
    sincos_(v[7], &s2, &c2);
    const R a1m2 = fmax(R(0), R(1) - N);
    const R a1m = sqrt_(a1m2);
    const cx<R> a1 = {a1m * c1, a1m * s1};
    // |c1|^2 = 1 - |a1|^2 - |b1|^2 = N - |b1|^2 (first column has unit norm).  Written with N, not with
    // 1 - (1 - N): the latter keeps N only to an absolute 1e-16 and loses log10(1/N) digits of c1 on links
    // close to the identity (measured on 8^4, eps = 0.01: link error 5.6e-12 -> 4.0e-16, R10).
    const R c1m = sqrt_(fmax(R(0), (N - b1.re * b1.re) - b1.im * b1.im));
    const cx<R> cc1 = {c1m * c2, c1m * s2};
    const R iN = R(1) / N;
    const cx<R> p = cmulc(a1, b1);        // conj(a1) b1
    const cx<R> q = cmulc(a1, cc1);       // conj(a1) c1
    // b2 = -(p a2 + conj(c1) conj(a3))/N ; b3 = (-p a3 + conj(c1) conj(a2))/N
    // c2 = (-q a2 + conj(b1) conj(a3))/N ; c3 = -(q a3 + conj(b1) conj(a2))/N
    const cx<R> pa2 = cmul(p, a2), pa3 = cmul(p, a3), qa2 = cmul(q, a2), qa3 = cmul(q, a3);
    const cx<R> c1a3 = conj_(cmul(cc1, a3)), c1a2 = conj_(cmul(cc1, a2));
    const cx<R> b1a3 = conj_(cmul(b1, a3)), b1a2 = conj_(cmul(b1, a2));
    u[0] = a1.re; u[1] = a1.im; u[2] = a2.re; u[3] = a2.im; u[4] = a3.re; u[5] = a3.im;
    u[6] = b1.re; u[7] = b1.im;
    u[8] = -(pa2.re + c1a3.re) * iN;  u[9] = -(pa2.im + c1a3.im) * iN;
    u[10] = (c1a2.re - pa3.re) * iN;  u[11] = (c1a2.im - pa3.im) * iN;
    u[12] = cc1.re; u[13] = cc1.im;
    u[14] = (b1a3.re - qa2.re) * iN;  u[15] = (b1a3.im - qa2.im) * iN;
    u[16] = -(qa3.re + b1a2.re) * iN; u[17] = -(qa3.im + b1a2.im) * iN;
  }
}

// Encode a full fp64 link into the stored RECON form (setup path, fp64 arithmetic).
template <int RECON>
LQ_DEV void compress_link(const double* __restrict__ u, double* __restrict__ v) {
  if constexpr (RECON == 18) {
#pragma unroll
    for (int k = 0; k < 18; ++k) v[k] = u[k];
  } else if constexpr (RECON == 12) {
#pragma unroll
    for (int k = 0; k < 12; ++k) v[k] = u[k];
  } else {
    v[0] = u[2]; v[1] = u[3]; v[2] = u[4]; v[3] = u[5]; v[4] = u[6]; v[5] = u[7];
    v[6] = atan2(u[1], u[0]);
    v[7] = atan2(u[13], u[12]);
  }
}

// convert RECON stored reals (fp64 values) into storage type of precision P
template <class P, int RECON>
LQ_DEV void quantize_link(const double* __restrict__ v, typename P::store_t* __restrict__ q) {
  if constexpr (!P::HALF) {
#pragma unroll
    for (int k = 0; k < RECON; ++k) q[k] = (typename P::store_t)v[k];
  } else {
#pragma unroll
    for (int k = 0; k < RECON; ++k) {
      double x = v[k];
      if (RECON == 8 && k >= 6) x *= (1.0 / 3.14159265358979323846);
      x = fmin(1.0, fmax(-1.0, x));
      q[k] = (short)(unsigned short)(__double2int_rn(x * 32767.0) + 32768);   // offset binary
    }
  }
}

// ---------------------------------------------------------------- index arithmetic
// Checkerboard index of one box: cb = xh + Xh*(y + Y*(z + Z*t)),  x = 2*xh + ((y+z+t+parity)&1).
// n / d with the precomputed m = ceil(2^32 / d) (d = 1 has no 32-bit m)
LQ_DEV int fast_div(int n, int d, unsigned m) { return d == 1 ? n : (int)__umulhi((unsigned)n, m); }
LQ_DEV void cb_to_coords(const Geom& g, int cb, int parity, int c[4]) {
  int r = fast_div(cb, g.Xh, g.mXh);
  const int xh = cb - r * g.Xh;
  int q = fast_div(r, g.X[1], g.mY);
  c[1] = r - q * g.X[1];
  c[3] = fast_div(q, g.X[2], g.mZ);
  c[2] = q - c[3] * g.X[2];
  c[0] = 2 * xh + ((c[1] + c[2] + c[3] + parity) & 1);
}
LQ_DEV int coords_to_cb(const Geom& g, const int c[4]) {
  return (c[0] >> 1) + g.Xh * (c[1] + g.X[1] * (c[2] + g.X[2] * c[3]));
}

}  // namespace lq
