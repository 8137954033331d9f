// mg_vm.cuh -- the shared-memory "wavefunction VM" kernel for g g -> t t~ + n g (sm_100a).
//
// One CTA evaluates E events for one assignment of the OUTER helicities and all assignments of the INNER
// helicities (see emitter/program.py).  The task program is produced by the emitter; this file holds the
// routines: external wavefunctions (PAPER.md:112-122 vxxxxx/oxxxxx/ixxxxx), off-shell wavefunctions
// (gluon<-gluon+gluon "VVV", gluon<-3 gluons "VVVV", quark<-quark+gluon "FFV"), closing
// amplitudes, colour-flow accumulation jamp += kappa*amp and the colour sum J^dagger C J
// (PAPER.md:136, 200).  Formulas: DESIGN.md "Feynman rules", chiral representation.
// All vertices are evaluated with g_s = 1; every diagram carries g_s^ng, applied once to |M_h|^2.
#pragma once
#include <cstdint>
#include <type_traits>
#include <cuda_runtime.h>

struct MgTask {              // 16 bytes: one work unit of one warp (a slice of a phase's packed item list of one routine)
  uint32_t w[4];
  // w0: type (4 bits) | sync << 4 (CTA barrier before this unit: first unit of a phase) | aux << 5 | first_only << 8
  // w1: i_begin, w2: i_end -- lane items [i_begin, i_end) of the list; lane item i = entry (i >> LOGE), event i & (E-1)
  //     (accumulation / channel units: first lane of the unit's 32-lane chunk, number of columns)
  // w3: first entry of the list in the index table (accumulation: unit id of the generated code; channel units: table offset)
  __host__ __device__ __forceinline__ uint32_t type() const { return w[0] & 15u; }
  __host__ __device__ __forceinline__ uint32_t sync() const { return (w[0] >> 4) & 1u; }
  __host__ __device__ __forceinline__ uint32_t aux() const { return (w[0] >> 5) & 7u; }
  __host__ __device__ __forceinline__ uint32_t first_only() const { return (w[0] >> 8) & 1u; }   // pass-invariant items (emitter/program.py)
  __host__ __device__ __forceinline__ uint32_t i_begin() const { return w[1]; }
  __host__ __device__ __forceinline__ uint32_t i_end() const { return w[2]; }
  __host__ __device__ __forceinline__ uint32_t tbl_off() const { return w[3]; }
};

struct MgProgramDesc {
  int ng, npar, ncolor, NC, nouter, nouter_legs, E, nthreads, nslot, ncol, ntasks, nidx, nacclist, colden, ndiag, namp, pos_t, pos_tb;
  long long flops_exec, flops_canonical;
  const MgTask* tasks; const uint16_t* idx; const uint32_t* acclist;
  const int16_t* colnum; const uint16_t* hin; const uint16_t* hout; const uint32_t* unitoff;
  // colnum is in jamp STORAGE-SLOT order; flowslot[slot] = colour flow stored there.  split = 1: flow and reversed flow sit ncolor / 2
  // slots apart and colprime is the block-diagonal matrix (Caa + Cab) (+) (Caa - Cab) of the J+- form (see the colour stage)
  const int16_t* colprime; const uint16_t* flowslot; int split;
};

enum { T_EXT = 0, T_VVV, T_VVVV, T_FFV, T_WCUR, T_AMP_DOT, T_AMP_FFV, T_AMP_VVV, T_AMP_VVVV, T_ACC, T_COMB, T_FFVR, T_QSUM, T_CHAN, T_VVVF, T_NOP = 15 };
__host__ __device__ __forceinline__ bool mg_table_unit(uint32_t type) { return type == T_ACC || type == T_CHAN; }   // units without index-table entries
// with this many outer-helicity passes or more, the passes of an event run back to back in one CTA: momenta, subset momenta and
// propagator denominators are staged once per event and (tensor-core colour stage) the external wavefunctions of the inner legs too
enum { MG_PER_TILE_MIN = 2 };
enum { MOMSTRIDE = 12 };     // per subset: K[4], 1/K^2, 1/(D + i m Gamma) re/im, pad, q = p_t - K [4]

struct VmArgs {
  const MgTask* tasks; const uint16_t* idx; const uint32_t* acclist;
  const void* colmat;        // TC numerators, blocked [row group][column][RPT rows] (see colour stage)
  const double* colfrag;     // FP64 tensor-core form: numerators of C' as m8n8k4 B fragments [non-zero block pair kb <= nb][k-step][32 lanes]
  const uint16_t* flowslot;  // [ncolor] colour flow stored in jamp slot s (the flow weights are written in flow order)
  const uint16_t* hin; const uint16_t* hout;
  const double* momenta; const double* gs;
  double* mh2;               // [nevt][ncomb]
  double* wpart;             // [nevt][nouter][ncolor]; [nevt][ncolor] when the outer passes of an event run in one CTA and the weights are summed on chip
  int nevt, layout, nwork;   // nwork = event tiles x outer helicity assignments
  int pos_t, pos_tb;         // bit positions of the t and t~ helicities inside the inner helicity combination
  uint32_t unitoff[33];      // work units of warp w: tasks[unitoff[w] .. unitoff[w+1])
  double mt, wt, gs_const, inv_colden;
  // Drell-Yan: couplings of the u quark and of the charged leptons to (photon, Z), each (left, right), then MZ, WZ
  double ew[10];
  unsigned int* counter;     // next work item (zeroed before the launch): the persistent CTAs share the batch dynamically
  // multichannel program only (CHAN instantiation of the kernel)
  const int* channel;        // [ceil(nevt / 32)] 1-based channel of every 32-event block, 0 = none; NULL = none
  const unsigned char* good; // [ncomb] good-helicity mask: the channel sums run over the good helicities
  double* chanpart;          // [nevt][nouter][NL / 32][2] partial (numerator, denominator) sums
};

// per-process compile-time configuration (emitted by emitter/emit.py)
template <int NG_, int NCOLOR_, int NC_, int E_, int NSLOT_, int NCOL_, int NT_, int MINB_, int NOUTER_LEGS_, int PID_ = NG_, int DY_ = 0> struct VmCfg {
  static constexpr int PID = PID_;      // program id: selects the generated accumulation code (a process may have a second, FP32, program)
  // DY = 1: Drell-Yan u(0) u~(1) -> e+(2) e-(3) + gluons (legs 4..).  NG then counts the labels on the quark line: the
  // gluons and, last, the gamma*/Z (a colourless block with a left- and a right-chiral current); massless line, no width.
  static constexpr bool DY = DY_ != 0;
  static constexpr int NGLUON = NG_ - DY_;
  static constexpr int NG = NG_, NPAR = NG_ + 2 + DY_, NCOLOR = NCOLOR_, NC = NC_, E = E_, NSLOT = NSLOT_, NCOL = NCOL_, NT = NT_, MINB = MINB_;
  static constexpr int NOUTER_LEGS = NOUTER_LEGS_, NOUTER = 1 << NOUTER_LEGS_, NCOMB = 1 << NPAR, NL = NC_ * E_, NSUB = 1 << NG_;
  static constexpr uint32_t STRIDE = (uint32_t)NSLOT_ * E_;
  static constexpr int ilog2(int x) { return x <= 1 ? 0 : 1 + ilog2(x >> 1); }
  static constexpr int LOGE = ilog2(E_), LOGNL = ilog2(NC_ * E_);
  static constexpr int G = NT_ / (NC_ * E_);                      // colour stage: row groups
  static constexpr int RPT = (NCOLOR_ + G - 1) / G;               // rows per thread
  static_assert((E_ & (E_ - 1)) == 0 && (NC_ & (NC_ - 1)) == 0, "E and NC must be powers of two");
  static_assert(NC_ * E_ <= NT_ && NT_ % (NC_ * E_) == 0 && NC_ * E_ >= 32, "NL must divide NT and cover a warp");
  static_assert(E_ <= 32, "E <= 32");
  // Colour sum on the FP64 tensor path (DMMA, mma.sync m8n8k4) where ncolor makes it a true GEMM (north_star): the jamp tile
  // of a work item is then 64 rows (32 helicity lanes x {re, im}) x NCOLOR, read as A fragments straight from shared memory.
  // To make those 8-byte gathers conflict-free the lane index of flow f is stored XOR SWZ(f) (a permutation inside the flow).
  static constexpr bool DMMA = NC_ * E_ == 32 && E_ == 1 && NCOLOR_ % 8 == 0 && NCOLOR_ >= 24;
  __host__ __device__ static constexpr uint32_t swz(uint32_t f) { return DMMA ? (((f & 1u) << 2) | (f & 2u)) : 0u; }
  // J+- form of the colour sum (DMMA only): C' is block diagonal with halves of HALF columns, so for a column block nb that lies
  // in the second half only the row blocks kb >= HALF / 8 are non-zero
  static constexpr int HALF = NCOLOR_ / 2;
  __host__ __device__ static constexpr int kb_lo(int nb) { return nb * 8 >= HALF ? HALF / 8 : 0; }
  // fragments stored before column block nb: sum over n < nb of (n - kb_lo(n) + 1), in closed form (called with a runtime nb)
  static constexpr int NB_FIRST_HI = (HALF + 7) / 8;              // first column block that lies in the second half
  __host__ __device__ static constexpr int frag_off(int nb) { return nb * (nb + 1) / 2 - (HALF / 8) * (nb > NB_FIRST_HI ? nb - NB_FIRST_HI : 0); }
};

template <class T> struct __align__(2 * sizeof(T)) Cx { T re, im; };
// D (8 x 8) += A (8 x 4, row) B (4 x 8, col) in FP64 on the tensor path: thread T holds A[T / 4][T % 4], B[T % 4][T / 4],
// D[T / 4][2 * (T % 4)] and D[T / 4][2 * (T % 4) + 1]
__device__ __forceinline__ void mg_dmma_f64(double& d0, double& d1, double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};" : "+d"(d0), "+d"(d1) : "d"(a), "d"(b));
}
// v with its sign flipped when signbit31 = 0x80000000 (0: unchanged)
__device__ __forceinline__ double flipsign(double v, uint32_t signbit31) {
  return __hiloint2double(__double2hiint(v) ^ (int)signbit31, __double2loint(v));
}
__device__ __forceinline__ float flipsign(float v, uint32_t signbit31) { return __uint_as_float(__float_as_uint(v) ^ signbit31); }
template <class T> __device__ __forceinline__ Cx<T> cmul(Cx<T> a, Cx<T> b) { return {a.re * b.re - a.im * b.im, a.re * b.im + a.im * b.re}; }
template <class T> __device__ __forceinline__ Cx<T> cadd(Cx<T> a, Cx<T> b) { return {a.re + b.re, a.im + b.im}; }
template <class T> __device__ __forceinline__ Cx<T> csub(Cx<T> a, Cx<T> b) { return {a.re - b.re, a.im - b.im}; }
template <class T> __device__ __forceinline__ Cx<T> cscale(T s, Cx<T> a) { return {s * a.re, s * a.im}; }
// a += b*c
template <class T> __device__ __forceinline__ void cfma(Cx<T>& a, Cx<T> b, Cx<T> c) {
  a.re = fma(b.re, c.re, a.re); a.re = fma(-b.im, c.im, a.re);
  a.im = fma(b.re, c.im, a.im); a.im = fma(b.im, c.re, a.im);
}
// Minkowski product of two complex 4-vectors (no conjugation)
template <class T> __device__ __forceinline__ Cx<T> mdot(const Cx<T>* a, const Cx<T>* b) {
  // two independent halves (shorter dependency chains): (a0 b0 - a1 b1) + (-a2 b2 - a3 b3)
  Cx<T> r = cmul(a[0], b[0]);
  Cx<T> q = cmul(cscale((T)-1, a[2]), b[2]);
  cfma(r, cscale((T)-1, a[1]), b[1]); cfma(q, cscale((T)-1, a[3]), b[3]);
  return cadd(r, q);
}
// real 4-vector . complex 4-vector
template <class T> __device__ __forceinline__ Cx<T> rdot(const T* k, const Cx<T>* a) {
  Cx<T> r;
  r.re = k[0] * a[0].re; r.re = fma(-k[1], a[1].re, r.re); r.re = fma(-k[2], a[2].re, r.re); r.re = fma(-k[3], a[3].re, r.re);
  r.im = k[0] * a[0].im; r.im = fma(-k[1], a[1].im, r.im); r.im = fma(-k[2], a[2].im, r.im); r.im = fma(-k[3], a[3].im, r.im);
  return r;
}

// wavefunction file: component-major, (re, im) interleaved: element (c, s) at wf[(c * STRIDE + s) * 2], so one 16-byte
// (8-byte in FP32) access per complex component and consecutive lanes = consecutive slots (conflict-free)
template <uint32_t STRIDE, class T> __device__ __forceinline__ void load_wf(const T* wf, uint32_t s, Cx<T>* w) {
  const Cx<T>* p = reinterpret_cast<const Cx<T>*>(wf) + s;
#pragma unroll
  for (int c = 0; c < 4; ++c) w[c] = p[c * STRIDE];
}
template <uint32_t STRIDE, class T> __device__ __forceinline__ void store_wf(T* wf, uint32_t s, const Cx<T>* w) {
  Cx<T>* p = reinterpret_cast<Cx<T>*>(wf) + s;
#pragma unroll
  for (int c = 0; c < 4; ++c) p[c * STRIDE] = w[c];
}

// row . slash(J):  slash(J) = [[0, J0 - J.sigma], [J0 + J.sigma, 0]]  (chiral representation)
template <class T> __device__ __forceinline__ void row_slash(const Cx<T>* a, const Cx<T>* J, Cx<T>* r) {
  Cx<T> Jp = cadd(J[0], J[3]), Jm = csub(J[0], J[3]);
  Cx<T> Jr = {J[1].re - J[2].im, J[1].im + J[2].re};   // J1 + i J2
  Cx<T> Jl = {J[1].re + J[2].im, J[1].im - J[2].re};   // J1 - i J2
  r[0] = cmul(a[2], Jp); cfma(r[0], a[3], Jr);
  r[1] = cmul(a[2], Jl); cfma(r[1], a[3], Jm);
  r[2] = cmul(a[0], Jm); cfma(r[2], cscale((T)-1, a[1]), Jr);
  r[3] = cmul(a[1], Jp); cfma(r[3], cscale((T)-1, a[0]), Jl);
}
// acc += (+-) row . slash(J).  The sign (bit 31 of sbit) is folded into J by sign-bit flips on the integer pipe and the products go
// straight into the accumulators: 8 additions + 32 FMA on the FP64 pipe instead of 8 + 32 + 8 with a separate signed accumulation.
template <class T> __device__ __forceinline__ void row_slash_acc(const Cx<T>* a, const Cx<T>* J, uint32_t sbit, Cx<T>* acc) {
  if constexpr (sizeof(T) == 4) {        // FP32 is bound by issue slots, not by the FMA pipe: the flips would cost more than the FMAs
    Cx<T> r[4];
    row_slash(a, J, r);
    const T sg = sbit ? (T)-1 : (T)1;
#pragma unroll
    for (int c = 0; c < 4; ++c) { acc[c].re = fma(sg, r[c].re, acc[c].re); acc[c].im = fma(sg, r[c].im, acc[c].im); }
    return;
  }
  Cx<T> K[4];
#pragma unroll
  for (int c = 0; c < 4; ++c) K[c] = {flipsign(J[c].re, sbit), flipsign(J[c].im, sbit)};
  Cx<T> Jp = cadd(K[0], K[3]), Jm = csub(K[0], K[3]);
  Cx<T> Jr = {K[1].re - K[2].im, K[1].im + K[2].re};   // J1 + i J2
  Cx<T> Jl = {K[1].re + K[2].im, K[1].im - K[2].re};   // J1 - i J2
  cfma(acc[0], a[2], Jp); cfma(acc[0], a[3], Jr);
  cfma(acc[1], a[2], Jl); cfma(acc[1], a[3], Jm);
  cfma(acc[2], a[0], Jm); cfma(acc[2], cscale((T)-1, a[1]), Jr);
  cfma(acc[3], a[1], Jp); cfma(acc[3], cscale((T)-1, a[0]), Jl);
}
// row . (slash(JL) P_L + slash(JR) P_R): the upper result components see JL, the lower ones JR (chiral representation)
template <class T> __device__ __forceinline__ void row_slash2(const Cx<T>* a, const Cx<T>* JL, const Cx<T>* JR, Cx<T>* r) {
  Cx<T> Lp = cadd(JL[0], JL[3]);
  Cx<T> Lr = {JL[1].re - JL[2].im, JL[1].im + JL[2].re}, Ll = {JL[1].re + JL[2].im, JL[1].im - JL[2].re};
  Cx<T> Lm = csub(JL[0], JL[3]);
  Cx<T> Rp = cadd(JR[0], JR[3]), Rm = csub(JR[0], JR[3]);
  Cx<T> Rr = {JR[1].re - JR[2].im, JR[1].im + JR[2].re}, Rl = {JR[1].re + JR[2].im, JR[1].im - JR[2].re};
  r[0] = cmul(a[2], Lp); cfma(r[0], a[3], Lr);
  r[1] = cmul(a[2], Ll); cfma(r[1], a[3], Lm);
  r[2] = cmul(a[0], Rm); cfma(r[2], cscale((T)-1, a[1]), Rr);
  r[3] = cmul(a[1], Rp); cfma(r[3], cscale((T)-1, a[0]), Rl);
}
// (slash(JL) P_L + slash(JR) P_R) . column: P_L keeps the upper column components, which feed the lower result components
template <class T> __device__ __forceinline__ void slash_col2(const Cx<T>* JL, const Cx<T>* JR, const Cx<T>* c, Cx<T>* r) {
  Cx<T> Rp = cadd(JR[0], JR[3]), Rm = csub(JR[0], JR[3]);
  Cx<T> Rr = {JR[1].re - JR[2].im, JR[1].im + JR[2].re}, Rl = {JR[1].re + JR[2].im, JR[1].im - JR[2].re};
  Cx<T> Lp = cadd(JL[0], JL[3]), Lm = csub(JL[0], JL[3]);
  Cx<T> Lr = {JL[1].re - JL[2].im, JL[1].im + JL[2].re}, Ll = {JL[1].re + JL[2].im, JL[1].im - JL[2].re};
  r[0] = cmul(Rm, c[2]); cfma(r[0], cscale((T)-1, Rl), c[3]);
  r[1] = cmul(Rp, c[3]); cfma(r[1], cscale((T)-1, Rr), c[2]);
  r[2] = cmul(Lp, c[0]); cfma(r[2], Ll, c[1]);
  r[3] = cmul(Lr, c[0]); cfma(r[3], Lm, c[1]);
}
// row . (slash(q) + m), q real
template <class T> __device__ __forceinline__ void row_slash_real_m(const Cx<T>* r, const T* q, T m, Cx<T>* s) {
  T qp = q[0] + q[3], qm = q[0] - q[3];
  Cx<T> qr = {q[1], q[2]}, ql = {q[1], -q[2]};
  s[0] = cscale(m, r[0]); s[0].re = fma(qp, r[2].re, s[0].re); s[0].im = fma(qp, r[2].im, s[0].im); cfma(s[0], r[3], qr);
  s[1] = cscale(m, r[1]); s[1].re = fma(qm, r[3].re, s[1].re); s[1].im = fma(qm, r[3].im, s[1].im); cfma(s[1], r[2], ql);
  s[2] = cscale(m, r[2]); s[2].re = fma(qm, r[0].re, s[2].re); s[2].im = fma(qm, r[0].im, s[2].im); cfma(s[2], cscale((T)-1, r[1]), qr);
  s[3] = cscale(m, r[3]); s[3].re = fma(qp, r[1].re, s[3].re); s[3].im = fma(qp, r[1].im, s[3].im); cfma(s[3], cscale((T)-1, r[0]), ql);
}
// slash(J) . column:  upper = (J0 - J.sigma) lower, lower = (J0 + J.sigma) upper
template <class T> __device__ __forceinline__ void slash_col(const Cx<T>* J, const Cx<T>* c, Cx<T>* r) {
  Cx<T> Jp = cadd(J[0], J[3]), Jm = csub(J[0], J[3]);
  Cx<T> Jr = {J[1].re - J[2].im, J[1].im + J[2].re};   // J1 + i J2
  Cx<T> Jl = {J[1].re + J[2].im, J[1].im - J[2].re};   // J1 - i J2
  r[0] = cmul(Jm, c[2]); cfma(r[0], cscale((T)-1, Jl), c[3]);
  r[1] = cmul(Jp, c[3]); cfma(r[1], cscale((T)-1, Jr), c[2]);
  r[2] = cmul(Jp, c[0]); cfma(r[2], Jl, c[1]);
  r[3] = cmul(Jr, c[0]); cfma(r[3], Jm, c[1]);
}
// (slash(q) + m) . column, q real
template <class T> __device__ __forceinline__ void slash_real_m_col(const T* q, T m, const Cx<T>* r, Cx<T>* s) {
  T qp = q[0] + q[3], qm = q[0] - q[3];
  Cx<T> qr = {q[1], q[2]}, ql = {q[1], -q[2]};
  s[0] = cscale(m, r[0]); s[0].re = fma(qm, r[2].re, s[0].re); s[0].im = fma(qm, r[2].im, s[0].im); cfma(s[0], cscale((T)-1, ql), r[3]);
  s[1] = cscale(m, r[1]); s[1].re = fma(qp, r[3].re, s[1].re); s[1].im = fma(qp, r[3].im, s[1].im); cfma(s[1], cscale((T)-1, qr), r[2]);
  s[2] = cscale(m, r[2]); s[2].re = fma(qp, r[0].re, s[2].re); s[2].im = fma(qp, r[0].im, s[2].im); cfma(s[2], ql, r[1]);
  s[3] = cscale(m, r[3]); s[3].re = fma(qm, r[1].re, s[3].re); s[3].im = fma(qm, r[1].im, s[3].im); cfma(s[3], qr, r[0]);
}
// W^mu = i (abar gamma^mu v)
template <class T> __device__ __forceinline__ void wcurrent(const Cx<T>* a, const Cx<T>* v, Cx<T>* W) {
  Cx<T> t0 = cmul(a[0], v[2]), t1 = cmul(a[1], v[3]), t2 = cmul(a[2], v[0]), t3 = cmul(a[3], v[1]);
  Cx<T> u0 = cmul(a[0], v[3]), u1 = cmul(a[1], v[2]), u2 = cmul(a[2], v[1]), u3 = cmul(a[3], v[0]);
  Cx<T> w0 = cadd(cadd(t0, t1), cadd(t2, t3));
  Cx<T> w1 = csub(cadd(u0, u1), cadd(u2, u3));
  Cx<T> w2i = cadd(csub(u1, u0), csub(u2, u3));        // W2 = i * w2i
  Cx<T> w3 = csub(csub(t0, t1), csub(t2, t3));
  // multiply by i: (re, im) -> (-im, re);  W2: i * (i w2i) = -w2i
  W[0] = {-w0.im, w0.re}; W[1] = {-w1.im, w1.re}; W[2] = {-w2i.re, -w2i.im}; W[3] = {-w3.im, w3.re};
}

// external wavefunctions from the raw momentum p = (E, px, py, pz), in the real type R: double in every mode except the
// all-FP32 one (the cancellation-prone scalars stay FP64 in the FP32 mode that is the default)
template <class R> __device__ __forceinline__ void ext_eps(const R* p, int lam, bool outgoing, Cx<R>* w) {
  R pt2 = p[1] * p[1] + p[2] * p[2];
  R pp = sqrt(pt2 + p[3] * p[3]);
  R pt = sqrt(pt2);
  R e1[4], e2[4];
  if (pt == (R)0) {
    e1[0] = 0; e1[1] = 1; e1[2] = 0; e1[3] = 0;
    e2[0] = 0; e2[1] = 0; e2[2] = p[3] >= 0 ? (R)1 : (R)-1; e2[3] = 0;
  } else {
    R inv = (R)1 / (pp * pt);
    e1[0] = 0; e1[1] = p[1] * p[3] * inv; e1[2] = p[2] * p[3] * inv; e1[3] = -pt2 * inv;
    e2[0] = 0; e2[1] = -p[2] / pt; e2[2] = p[1] / pt; e2[3] = 0;
  }
  const R s = (R)0.70710678118654752440;
  R sg = outgoing ? (R)1 : (R)-1;   // eps* for outgoing gluons
#pragma unroll
  for (int m = 0; m < 4; ++m) { w[m].re = -(R)lam * e1[m] * s; w[m].im = sg * e2[m] * s; }
}
template <class R> __device__ __forceinline__ void ext_chi(const R* p, R pp, int lam, Cx<R>* x) {
  if (pp + p[3] <= (R)0 || (p[1] == (R)0 && p[2] == (R)0 && p[3] < (R)0)) {
    if (lam > 0) { x[0] = {0, 0}; x[1] = {1, 0}; } else { x[0] = {-1, 0}; x[1] = {0, 0}; }
    return;
  }
  // near the -z axis |p| + p_z cancels: use p_T^2 / (|p| - p_z) there (the same number, all digits kept)
  const R s = p[3] >= (R)0 ? pp + p[3] : fma(p[1], p[1], p[2] * p[2]) / (pp - p[3]);
  R N = (R)1 / sqrt(2 * pp * s);
  if (lam > 0) { x[0] = {N * s, 0}; x[1] = {N * p[1], N * p[2]}; }
  else { x[0] = {-N * p[1], N * p[2]}; x[1] = {N * s, 0}; }
}
// kind 2: ubar(p, lam) row spinor of an outgoing fermion; kind 3: v(p, lam) column spinor of an outgoing antifermion
template <class R> __device__ __forceinline__ void ext_spinor(const R* p, R m, int lam, int kind, Cx<R>* w) {
  R pp = sqrt(p[1] * p[1] + p[2] * p[2] + p[3] * p[3]);
  R wp, wm;
  if (m == (R)0) { wp = sqrt(2 * pp); wm = 0; } else { wp = sqrt(p[0] + pp); wm = m / wp; }
  Cx<R> x[2];
  if (kind == 2) {
    ext_chi(p, pp, lam, x);
    R wup = lam > 0 ? wm : wp, wlo = lam > 0 ? wp : wm;
    // u = (wup x ; wlo x);  ubar = u^dagger gamma^0 = (conj(u2), conj(u3), conj(u0), conj(u1))
    w[0] = {wlo * x[0].re, -wlo * x[0].im}; w[1] = {wlo * x[1].re, -wlo * x[1].im};
    w[2] = {wup * x[0].re, -wup * x[0].im}; w[3] = {wup * x[1].re, -wup * x[1].im};
  } else {
    ext_chi(p, pp, -lam, x);
    R l = (R)lam;
    R wl = lam > 0 ? wp : wm, wml = lam > 0 ? wm : wp;
    w[0] = {-l * wl * x[0].re, -l * wl * x[0].im}; w[1] = {-l * wl * x[1].re, -l * wl * x[1].im};
    w[2] = {l * wml * x[0].re, l * wml * x[0].im}; w[3] = {l * wml * x[1].re, l * wml * x[1].im};
  }
}

// Drell-Yan: the gamma*/Z as seen by a quark line of chirality chi (0 left, 1 right):
//   J^mu = sum_V g^q_{V,chi} / (s_ll - M_V^2 + i M_V W_V) * ubar(e-, h3) gamma^mu (g^l_{V,L} P_L + g^l_{V,R} P_R) v(e+, h2)
// so that its vertex on the line is i slash(J), like a gluon's with g_s = 1 (electroweak part).
// ew[] = u-quark couplings (photon L, R, Z L, R), lepton couplings (photon L, R, Z L, R), MZ, WZ.
template <class R> __device__ __forceinline__ void ext_ew_current(const R* pep, const R* pem, int hep, int hem, int chi, const double* ew, Cx<R>* J) {
  Cx<R> a[4], v[4];
  ext_spinor<R>(pem, (R)0, hem, 2, a);                       // ubar of the outgoing e-
  ext_spinor<R>(pep, (R)0, hep, 3, v);                       // v of the outgoing e+
  // abar gamma^mu P_L v uses (a2, a3; v0, v1), abar gamma^mu P_R v uses (a0, a1; v2, v3)
  Cx<R> jL[4], jR[4];
  {
    Cx<R> t2 = cmul(a[2], v[0]), t3 = cmul(a[3], v[1]), u2 = cmul(a[2], v[1]), u3 = cmul(a[3], v[0]);
    jL[0] = cadd(t2, t3); jL[1] = cscale((R)-1, cadd(u2, u3));
    Cx<R> d = csub(u2, u3); jL[2] = {-d.im, d.re};           // i (a2 v1 - a3 v0)
    jL[3] = csub(t3, t2);
    Cx<R> t0 = cmul(a[0], v[2]), t1 = cmul(a[1], v[3]), u0 = cmul(a[0], v[3]), u1 = cmul(a[1], v[2]);
    jR[0] = cadd(t0, t1); jR[1] = cadd(u0, u1);
    Cx<R> e = csub(u1, u0); jR[2] = {-e.im, e.re};           // i (a1 v2 - a0 v3)
    jR[3] = csub(t0, t1);
  }
  // s_ll = 2 p_e+.p_e- of two massless momenta: nearly collinear leptons would lose their digits in E E' - p.p', so in the same half
  // space the product is |p x p'|^2 / (E E' + p.p') (reading 6; the photon pole 1 / s_ll amplifies the error)
  R sll;
  {
    const R ee = pep[0] * pem[0], d3 = pep[1] * pem[1] + pep[2] * pem[2] + pep[3] * pem[3];
    sll = ee - d3;
    if ((ee > 0) == (d3 > 0)) {
      const R cx = pep[2] * pem[3] - pep[3] * pem[2], cy = pep[3] * pem[1] - pep[1] * pem[3], cz = pep[1] * pem[2] - pep[2] * pem[1];
      sll = (cx * cx + cy * cy + cz * cz) / (ee + d3);
    }
    sll *= 2;
  }
  const R dz = sll - (R)(ew[8] * ew[8]), gz = (R)(ew[8] * ew[9]), nz = dz * dz + gz * gz;
  // 1 / s_ll and 1 / (dz + i gz) = (dz - i gz) / nz, times the quark coupling of this chirality
  const Cx<R> cA = {(R)ew[chi] / sll, (R)0}, cZ = {(R)ew[2 + chi] * dz / nz, -(R)ew[2 + chi] * gz / nz};
#pragma unroll
  for (int m = 0; m < 4; ++m) {
    const Cx<R> la = cadd(cscale((R)ew[4], jL[m]), cscale((R)ew[5], jR[m]));
    const Cx<R> lz = cadd(cscale((R)ew[6], jL[m]), cscale((R)ew[7], jR[m]));
    J[m] = cmul(cA, la); cfma(J[m], cZ, lz);
  }
}

// ---- software-pipelined loads of the read-only program tables (L2-resident, streamed) --------------------------
// a warp fetches 32 of its unit descriptors at once (one per lane) and broadcasts them by shuffle
struct UnitBatch {
  uint4 lo;
  __device__ __forceinline__ void load(const MgTask* tasks, uint32_t first, uint32_t end, uint32_t lane) {
    const uint32_t u = first + lane < end ? first + lane : end - 1;
    lo = __ldg(reinterpret_cast<const uint4*>(tasks + u));
  }
  __device__ __forceinline__ MgTask get(uint32_t k) const {
    MgTask t;
    t.w[0] = __shfl_sync(0xffffffffu, lo.x, k); t.w[1] = __shfl_sync(0xffffffffu, lo.y, k);
    t.w[2] = __shfl_sync(0xffffffffu, lo.z, k); t.w[3] = __shfl_sync(0xffffffffu, lo.w, k);
    return t;
  }
};
// 16-byte index-table entry of lane item i of a unit: eight 16-bit fields
//   u0..u3 operand slots (absolute), u4 result slot or helicity-combination base, u5 = mA | mB << 8 (gluon-subset masks
//   or bit positions), u6 amplitude-buffer column, u7 flags.  All same-type tasks of a phase share one packed item list.
// accumulation units generated by the emitter (specialised per process in generated/mg_programs.inc)
// run(unit, ab, jq0..jq3): ab = amplitude buffer at this lane, jq[f & 3] = jamp at this lane's (swizzled) position for flow f
template <int PID, class T> struct MgAcc { static __device__ __forceinline__ void run(uint32_t, const Cx<T>*, Cx<T>*, Cx<T>*, Cx<T>*, Cx<T>*) {} };
// false when the generated units start every flow from zero themselves (then jamp needs no zero fill per work item)
template <int PID> struct MgAccZeroFill { static constexpr bool value = true; };

// Table form of an accumulation unit, for processes whose generated code would not fit the instruction cache (every
// unit's code runs once per work item, so straight-line code is bound by instruction-fetch latency there).  tbl is a
// __constant__ array: [number of flows] then per flow [jamp offset | pairs << 20][pairs x (amplitude offset | sign << 31)],
// offsets in complex elements.  What is left of kappa after the phase convention of the currents is a sign.
#define MG_TBL(p) (*(p))
template <class T> __device__ __forceinline__ void mg_acc_one(const uint32_t e, const Cx<T>* __restrict__ ab, Cx<T>& j) {
  const Cx<T> v = ab[e & 0xffffu];
  const uint32_t sg = e & 0x80000000u;
  j.re += flipsign(v.re, sg); j.im += flipsign(v.im, sg);
}
template <class T> __device__ __forceinline__ void mg_acc_table(const uint32_t* __restrict__ tbl, uint32_t p,
                                                                 const Cx<T>* __restrict__ ab, Cx<T>* __restrict__ jl) {
  const uint32_t nfl = MG_TBL(tbl + p); ++p;
  for (uint32_t f = 0; f < nfl; ++f) {
    const uint32_t h = MG_TBL(tbl + p), np = h >> 20; ++p;
    Cx<T>* jp = jl + (h & 0xfffffu);
    Cx<T> j = *jp;
    uint32_t q = 0;
    for (; q + 4 <= np; q += 4) {
      const uint32_t e0 = MG_TBL(tbl + p + q), e1 = MG_TBL(tbl + p + q + 1), e2 = MG_TBL(tbl + p + q + 2), e3 = MG_TBL(tbl + p + q + 3);
      mg_acc_one(e0, ab, j); mg_acc_one(e1, ab, j); mg_acc_one(e2, ab, j); mg_acc_one(e3, ab, j);
    }
    for (; q < np; ++q) mg_acc_one(MG_TBL(tbl + p + q), ab, j);
    p += np;
    *jp = j;
  }
}

template <class CFG> __device__ __forceinline__ uint4 ld_entry(const VmArgs& a, const MgTask& t, uint32_t i) {
  return __ldg(reinterpret_cast<const uint4*>(a.idx) + t.tbl_off() + (i >> CFG::LOGE) * (t.type() == T_QSUM ? 3u : 1u));   // QSUM: 48-byte entries
}
#define MG_U0(r) ((r).x & 0xffffu)
#define MG_U1(r) ((r).x >> 16)
#define MG_U2(r) ((r).y & 0xffffu)
#define MG_U3(r) ((r).y >> 16)
#define MG_U4(r) ((r).z & 0xffffu)
#define MG_U5(r) ((r).z >> 16)
#define MG_U6(r) ((r).w & 0xffffu)
#define MG_U7(r) ((r).w >> 16)

// item loop of one warp over its unit, with the next entry prefetched one iteration ahead
template <class CFG, class F>
__device__ __forceinline__ void for_items(const VmArgs& a, const MgTask& tk, uint32_t nlane, uint32_t i0, uint4 raw0, F f) {
  uint32_t i = i0; uint4 raw = raw0;
  while (i < nlane) {
    uint32_t in = i + 32;
    uint4 rn = raw;
    if (in < nlane) rn = ld_entry<CFG>(a, tk, in);
    f(i, raw);
    i = in; raw = rn;
  }
}

// FP32 wavefunctions need half the shared memory and registers: ask for more resident CTAs.  Measured on B200 (round 2): twice as
// many for the FP32 program of gg->ttgg (12.4 vs 18.1 ms) and for Drell-Yan; 1.5 times for gg->tt~ and gg->tt~g, where the
// 64-register cap of the doubled count spills (gg->ttg 2.70 vs 3.11 ms, gg->tt 0.51 vs 0.56); not for gg->ttggg (one CTA per SM).
template <class T, class CFG> constexpr int mg_min_blocks() {
  if (sizeof(T) != 4 || CFG::NG >= 5) return CFG::MINB;
  return (CFG::DY || CFG::NG == 4) ? 2 * CFG::MINB : 3 * CFG::MINB / 2;
}

// T: wavefunctions / amplitudes / jamp, TC: colour sum, TS: external wavefunctions, subset momenta and propagator denominators
// (double in every mode except the all-FP32 one)
template <class T, class TC, class CFG, bool CHAN = false, class TS = double>
__global__ void __launch_bounds__(CFG::NT, mg_min_blocks<T, CFG>()) mg_vm_kernel(const VmArgs a) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  constexpr int E = CFG::E, NL = CFG::NL, NT = CFG::NT, NG = CFG::NG, NPAR = CFG::NPAR, NCOLOR = CFG::NCOLOR;
  constexpr uint32_t STRIDE = CFG::STRIDE;
  const uint32_t tid = threadIdx.x;
  double* praw = reinterpret_cast<double*>(smem_raw);       // [8][4][E] raw momenta (double)
  double* gsE = praw + 8 * 4 * E;                           // [E]
  double* red = gsE + ((E + 1) & ~1);                       // [NT] reduction scratch of the colour stage (keeps wf 16-byte aligned)
  T* mom = reinterpret_cast<T*>(red + NT);                  // [NSUB][MOMSTRIDE][E]; kept for all outer-helicity passes of an event tile
  T* wf = mom + CFG::NSUB * MOMSTRIDE * E;                  // [8][NSLOT*E]
  T* ampbuf = wf + 8 * STRIDE;                              // [NCOL + 1][NL][2] (last column: zeros)
  T* jamp = ampbuf + (CFG::NCOL + 1) * 2 * NL;              // [NCOLOR][NL][2]; last, so that wf|ampbuf is one dead block at the colour stage
  Cx<T>* amp2 = reinterpret_cast<Cx<T>*>(ampbuf);           // both as (re, im) pairs: one 128-bit (FP64) access per complex number
  Cx<T>* jamp2 = reinterpret_cast<Cx<T>*>(jamp);
  // multichannel program: no jamp; in its place the channel sums [2][NL] (numerator, denominator) of the current pass
  double* chansum = reinterpret_cast<double*>(jamp);
  __shared__ int s_chan[32];                                // channel of the tile's events
  __shared__ Cx<T> s_extside[2][2][4];                      // polarisation vectors of the outer legs for both helicities (first pass)
  __shared__ int s_extslot[2];                              // and the wavefunction slots they belong to

  // persistent CTAs: each walks the (event tile, outer helicity) work items with a grid stride; the outer-helicity passes
  // of a tile run back to back in one CTA (raw momenta, subset momenta and propagator denominators staged once per tile)
  // when there are four of them (measured on B200: +3% gg->ttggg, -4% gg->ttgg with its two passes and four CTAs per SM)
  constexpr bool PER_TILE = CFG::NOUTER >= MG_PER_TILE_MIN;
  // the external wavefunctions survive from one outer pass of an event to the next when nothing overwrites the wavefunction file
  // in between: the tensor-core colour stage streams its matrix from global memory (the other form stages it in the dead file)
  constexpr bool KEEP_EXT = PER_TILE && E == 1 && CFG::NOUTER_LEGS <= 2 && CFG::DMMA && !CHAN && std::is_same<T, double>::value && std::is_same<TC, double>::value;
  const int nloop = PER_TILE ? a.nwork / CFG::NOUTER : a.nwork;
  // items are handed out by a device-wide counter: SMs that run slower (instruction-cache and clock differences between
  // GPCs) take fewer items instead of holding the launch up
  // (the two small processes keep the static grid stride: their items are too short to pay for the counter)
  constexpr bool DYNAMIC = NG >= 4;
  __shared__ int s_item;
  for (int static_item = blockIdx.x;; static_item += gridDim.x) {
  if (DYNAMIC) {
    if (tid == 0) s_item = (int)atomicAdd(a.counter, 1u);
    __syncthreads();
  }
  const int item = DYNAMIC ? s_item : static_item;       // (s_item is rewritten only after the barriers of this item's passes)
  if (item >= nloop) break;
  double wacc = 0;         // colour-flow weight of this thread's flow, summed over the passes of the tile (E = 1 form)
  for (int pass = 0; pass < (PER_TILE ? CFG::NOUTER : 1); ++pass) {
  const int work = PER_TILE ? item * CFG::NOUTER + pass : item;
  const int tile = work / CFG::NOUTER, outer = work % CFG::NOUTER;
  const long long ev0 = (long long)tile * E;
  const bool stage = !PER_TILE || pass == 0;

  // this warp's work-unit list; prefetch the first descriptors while staging
  const uint32_t lane = tid & 31, warp = tid >> 5;
  const uint32_t u_begin = a.unitoff[warp], u_end = a.unitoff[warp + 1];
  UnitBatch batch;
  batch.load(a.tasks, u_begin, u_end, lane);

  // ---- stage raw momenta ------------------------------------------------------------------------------------
  if (stage)
  for (int i = tid; i < NPAR * 4 * E; i += NT) {
    int e = i % E, c = (i / E) % 4, leg = i / (4 * E);
    long long ev = ev0 + e; if (ev >= a.nevt) ev = a.nevt - 1;
    double v;
    if (a.layout == 0) v = a.momenta[(ev * NPAR + leg) * 4 + c];
    else v = a.momenta[(((ev >> 5) * NPAR + leg) * 4 + c) * 32 + (ev & 31)];
    praw[(leg * 4 + c) * E + e] = v;
  }
  if (stage)
  for (int e = tid; e < E; e += NT) {
    long long ev = ev0 + e; if (ev >= a.nevt) ev = a.nevt - 1;
    gsE[e] = a.gs ? a.gs[ev] : a.gs_const;
    if (CHAN) s_chan[e] = a.channel ? a.channel[ev >> 5] : 0;
  }
  if (KEEP_EXT && pass > 0 && tid < CFG::NOUTER_LEGS * 4) {
    const int k = (int)tid >> 2, c = (int)tid & 3, bit = (outer >> (CFG::NOUTER_LEGS - 1 - k)) & 1;
    reinterpret_cast<Cx<T>*>(wf)[(uint32_t)c * STRIDE + (uint32_t)s_extslot[k]] = s_extside[k][bit][c];
  }
  if (CHAN) {
    for (int i = tid; i < 2 * NL; i += NT) chansum[i] = 0.0;
  } else if (MgAccZeroFill<CFG::PID>::value)
    for (int i = tid; i < NCOLOR * 2 * NL; i += NT) jamp[i] = (T)0;
  for (int i = tid; i < 2 * NL; i += NT) ampbuf[CFG::NCOL * 2 * NL + i] = (T)0;      // zero column for padded accumulation entries
  __syncthreads();
  // ---- per-event subset momenta and propagator denominators, in double -----
  if (stage)
  for (int i = tid; i < CFG::NSUB * E; i += NT) {
    int e = i % E, S = i / E;
    TS K[4] = {0, 0, 0, 0}, K2 = 0, D = 0;
    TS p2[4];
    if constexpr (CFG::DY) {
      // labels g < NGLUON: outgoing gluons (legs 4 + g, k = -p); label NGLUON: the gamma*/Z, k_V = -(p_e+ + p_e-), k_V^2 = 2 p_e+.p_e-;
      // the momentum carried along the quark line at its row end is -p_u~
#pragma unroll
      for (int c = 0; c < 4; ++c) p2[c] = -(TS)praw[(1 * 4 + c) * E + e];
      TS kk[NG][4];
#pragma unroll
      for (int g = 0; g < NG; ++g)
#pragma unroll
        for (int c = 0; c < 4; ++c)
          kk[g][c] = g < CFG::NGLUON ? -(TS)praw[((4 + g) * 4 + c) * E + e] : -((TS)praw[(2 * 4 + c) * E + e] + (TS)praw[(3 * 4 + c) * E + e]);
      // 2 x.y; two massless momenta in the same half space (x0 y0 and x.y of one sign) take the cancellation-free form
      // |x x y|^2 / (x0 y0 + x.y) (reading 6)
      auto pair2 = [](const TS* x, const TS* y, bool massless) -> TS {
        const TS ee = x[0] * y[0], d3 = x[1] * y[1] + x[2] * y[2] + x[3] * y[3];
        TS r = ee - d3;
        if (massless && (ee > 0) == (d3 > 0)) {
          const TS cx = x[2] * y[3] - x[3] * y[2], cy = x[3] * y[1] - x[1] * y[3], cz = x[1] * y[2] - x[2] * y[1];
          r = (cx * cx + cy * cy + cz * cz) / (ee + d3);
        }
        return 2 * r;
      };
      auto k2of = [&](int M) -> TS {
        TS s = 0;
#pragma unroll
        for (int g = 0; g < NG; ++g) {
          if (!(M >> g & 1)) continue;
          if (g == CFG::NGLUON) {
            TS pa[4], pb[4];
#pragma unroll
            for (int c = 0; c < 4; ++c) { pa[c] = (TS)praw[(2 * 4 + c) * E + e]; pb[c] = (TS)praw[(3 * 4 + c) * E + e]; }
            s += pair2(pa, pb, true);              // the leptons are massless too
          }
#pragma unroll
          for (int h = g + 1; h < NG; ++h)
            if (M >> h & 1) s += pair2(kk[g], kk[h], h < CFG::NGLUON);
        }
        return s;
      };
#pragma unroll
      for (int g = 0; g < NG; ++g) {
        if (!(S >> g & 1)) continue;
#pragma unroll
        for (int c = 0; c < 4; ++c) K[c] += kk[g][c];
      }
      K2 = k2of(S);
      // By momentum conservation -p_u~ - K_S = p_u + K_Sc (Sc: the other labels), both ends of the line massless: the denominator is
      // taken from the side with fewer labels, so that a gluon collinear with the incoming quark gives one small product instead of
      // a sum of O(s) terms that cancel
      // (a tie goes to the side without the boson: all its products are then of massless momenta)
      if (2 * __popc(S) > NG || (2 * __popc(S) == NG && (S >> CFG::NGLUON & 1))) {
        const int Sc = ((1 << NG) - 1) ^ S;
        TS p1[4];
#pragma unroll
        for (int c = 0; c < 4; ++c) p1[c] = (TS)praw[(0 * 4 + c) * E + e];
        D = k2of(Sc);
#pragma unroll
        for (int g = 0; g < NG; ++g)
          if (Sc >> g & 1) D += pair2(p1, kk[g], g < CFG::NGLUON);
      } else {
        D = K2;
#pragma unroll
        for (int g = 0; g < NG; ++g)
          if (S >> g & 1) D -= pair2(p2, kk[g], g < CFG::NGLUON);
      }
    } else {
#pragma unroll
    for (int c = 0; c < 4; ++c) p2[c] = (TS)praw[(2 * 4 + c) * E + e];
#pragma unroll
    for (int g = 0; g < NG; ++g) {
      if (!(S >> g & 1)) continue;
      const int lg = g < 2 ? g : g + 2; const TS sg = g < 2 ? (TS)1 : (TS)-1;
      TS kg[4];
#pragma unroll
      for (int c = 0; c < 4; ++c) { kg[c] = sg * (TS)praw[(lg * 4 + c) * E + e]; K[c] += kg[c]; }
#pragma unroll
      for (int h = g + 1; h < NG; ++h) {
        if (!(S >> h & 1)) continue;
        const int lh = h < 2 ? h : h + 2; const TS sh = h < 2 ? (TS)1 : (TS)-1;
        TS kh[4];
#pragma unroll
        for (int c = 0; c < 4; ++c) kh[c] = sh * (TS)praw[(lh * 4 + c) * E + e];
        // 2 k_g.k_h of two massless momenta.  Nearly collinear gluons would lose their digits in E_g E_h - k_g.k_h, so where both
        // terms have the same sign the product is taken as |k_g x k_h|^2 / (E_g E_h + k_g.k_h) (equal for k^2 = 0)
        const TS ee = kg[0] * kh[0], d3 = kg[1] * kh[1] + kg[2] * kh[2] + kg[3] * kh[3];
        TS gh = ee - d3;
        if ((ee > 0) == (d3 > 0)) {
          const TS cx = kg[2] * kh[3] - kg[3] * kh[2], cy = kg[3] * kh[1] - kg[1] * kh[3], cz = kg[1] * kh[2] - kg[2] * kh[1];
          gh = (cx * cx + cy * cy + cz * cz) / (ee + d3);
        }
        K2 += 2 * gh;
      }
    }
    D = K2;
#pragma unroll
    for (int g = 0; g < NG; ++g) {
      if (!(S >> g & 1)) continue;
      const int lg = g < 2 ? g : g + 2; const TS sg = g < 2 ? (TS)1 : (TS)-1;
      TS kg[4];
#pragma unroll
      for (int c = 0; c < 4; ++c) kg[c] = sg * (TS)praw[(lg * 4 + c) * E + e];
      D -= 2 * (p2[0] * kg[0] - p2[1] * kg[1] - p2[2] * kg[2] - p2[3] * kg[3]);
    }
    }
    T* m = mom + (size_t)S * MOMSTRIDE * E + e;
#pragma unroll
    for (int c = 0; c < 4; ++c) { m[c * E] = (T)K[c]; m[(8 + c) * E] = (T)(p2[c] - K[c]); }
    m[4 * E] = (T)((S & (S - 1)) ? (TS)1 / K2 : (TS)0);
    const TS gw = (TS)a.mt * (TS)a.wt, nrm = D * D + gw * gw;
    m[5 * E] = (T)(S ? D / nrm : (TS)0); m[6 * E] = (T)(S ? -gw / nrm : (TS)0); m[7 * E] = (T)0;
  }

  // ---- task program -------------------------------------------------------------------------------------------
  const T mt = (T)a.mt;
  MgTask tk = batch.get(0), tk1 = tk;
  uint32_t batch_first = u_begin;
  uint32_t i0 = tk.i_begin() + lane;
  uint32_t nlane = tk.i_end();
  uint4 raw0 = make_uint4(0, 0, 0, 0);
  if (!mg_table_unit(tk.type()) && i0 < nlane) raw0 = ld_entry<CFG>(a, tk, i0);
  for (uint32_t it = u_begin; it < u_end; ++it) {
    // next unit's descriptor (from the batch) and the first table entry of the next unit
    uint32_t i0n = 0, nlanen = 0;
    uint4 raw0n = make_uint4(0, 0, 0, 0);
    if (it + 1 < u_end) {
      if (it + 1 - batch_first == 32) { batch_first = it + 1; batch.load(a.tasks, batch_first, u_end, lane); }
      tk1 = batch.get(it + 1 - batch_first);
      i0n = tk1.i_begin() + lane; nlanen = tk1.i_end();
      if (!mg_table_unit(tk1.type()) && i0n < nlanen) raw0n = ld_entry<CFG>(a, tk1, i0n);
    }
    if (tk.sync()) __syncthreads();
    __syncwarp();      // a warp's units run in order: the closing sums of a flow follow its accumulation unit in the same warp (other lanes)
    // units whose results depend on no outer leg: the first outer-helicity pass of the event left them in the wavefunction file
    const bool skip_unit = KEEP_EXT && pass > 0 && tk.first_only();
    if (!skip_unit && (i0 < nlane || mg_table_unit(tk.type()))) {
      switch (tk.type()) {
        case T_CHAN: {
          // multichannel sums: this warp's 32 lanes add |A|^2 of every pending amplitude column (one column
          // = one diagram without four-gluon vertices = one channel) into their denominator and, where the column is the
          // channel of the lane's event, numerator.  One unit per lane chunk per phase: no two warps touch the same sums.
          if constexpr (CHAN) {
            const uint32_t l = tk.i_begin() + lane, ncols = tk.i_end();
            const uint32_t* tb = a.acclist + tk.tbl_off();
            const uint32_t mych = (uint32_t)s_chan[l & (E - 1)];
            double num = 0, den = 0;
            for (uint32_t c = 0; c < ncols; ++c) {
              const uint32_t id = __ldg(tb + c);
              const Cx<T> v = amp2[c * NL + l];
              const double d = fma((double)v.re, (double)v.re, (double)v.im * (double)v.im);
              den += d;
              num += id == mych ? d : 0.0;
            }
            chansum[l] += num; chansum[NL + l] += den;
          }
        } break;
        case T_ACC: {
          // One unit = a group of colour flows x 32 lanes of one warp: jamp[flow][l] += sum of kappa * ampbuf[col][l].  The
          // code is generated per unit by the emitter (generated/mg_programs.inc, MgAcc<NG, T>): buffer offsets and the
          // signs of kappa in {1, i, -1, -i} are immediates, so a pair costs one (re, im) shared-memory load and two adds.
          const uint32_t l = tk.i_begin() + lane;
          MgAcc<CFG::PID, T>::run(tk.tbl_off(), amp2 + l, jamp2 + (l ^ CFG::swz(0)), jamp2 + (l ^ CFG::swz(1)), jamp2 + (l ^ CFG::swz(2)), jamp2 + (l ^ CFG::swz(3)));
        } break;
        case T_EXT: {
          for_items<CFG>(a, tk, nlane, i0, raw0, [&](uint32_t i, uint4 raw) {
            const uint32_t e = i & (E - 1);
            const int leg = MG_U0(raw), code = MG_U1(raw), kind = MG_U2(raw);
            // The wavefunctions of the inner legs do not depend on the pass.  Where the outer passes of an event run back to back and
            // nothing overwrites the wavefunction file in between (the tensor-core colour stage streams its matrix from global memory),
            // they are computed in the first pass only: this single-warp phase cost 13% of the g g -> t t~ g g g kernel.
            // The outer legs' polarisation vectors are computed for both helicities in the first pass (side buffer) and copied into
            // their slots at the start of the later passes, so this phase does no arithmetic after the first pass.
            if (KEEP_EXT && pass > 0) return;
            const int bit = code < 2 ? code : ((outer >> (CFG::NOUTER_LEGS - 1 - (code - 2))) & 1);
            const int lam = bit ? 1 : -1;
            TS p[4];
#pragma unroll
            for (int c = 0; c < 4; ++c) p[c] = (TS)praw[(leg * 4 + c) * E + e];
            Cx<TS> w[4];
            // (the g g -> t t~ kernels keep the plain two-way branch: with a third arm the compiler spilled in the 128-register
            // kernel of g g -> t t~ g g g and it ran 4% slower, 68.7 vs 66.0 ms on B200)
            if constexpr (!CFG::DY) { if (kind < 2) ext_eps<TS>(p, lam, kind == 1, w); else ext_spinor<TS>(p, (TS)a.mt, lam, kind, w); }
            else if (kind < 2) ext_eps<TS>(p, lam, kind == 1, w);
            else if (kind < 4) ext_spinor<TS>(p, (TS)a.mt, lam, kind, w);
            else {
              if (kind < 6) {
                // 4: vbar(p, lam) of the incoming antiquark = bar of v; 5: u(p, lam) of the incoming quark = bar^-1 of ubar
                Cx<TS> x[4];
                ext_spinor<TS>(p, (TS)0, lam, kind == 4 ? 3 : 2, x);
                w[0] = {x[2].re, -x[2].im}; w[1] = {x[3].re, -x[3].im}; w[2] = {x[0].re, -x[0].im}; w[3] = {x[1].re, -x[1].im};
              } else {
                // 6 / 7: the gamma*/Z current for a left- / right-chiral quark line; helicity codes of e+ (u1) and e- (u3)
                TS pep[4], pem[4];
#pragma unroll
                for (int c = 0; c < 4; ++c) { pep[c] = (TS)praw[(2 * 4 + c) * E + e]; pem[c] = (TS)praw[(3 * 4 + c) * E + e]; }
                ext_ew_current<TS>(pep, pem, lam, MG_U3(raw) ? 1 : -1, kind - 6, a.ew, w);
              }
            }
            Cx<T> o[4];
#pragma unroll
            for (int c = 0; c < 4; ++c) o[c] = {(T)w[c].re, (T)w[c].im};
            store_wf<STRIDE>(wf, MG_U4(raw) * E + e, o);
            if (KEEP_EXT && code >= 2) {
              // eps(-lam) = -conj(eps(lam)) for the same in/out kind: w(lam) = (-lam e1 + i sg e2) / sqrt(2)
              const int k = code - 2;
              s_extslot[k] = (int)MG_U4(raw);
#pragma unroll
              for (int c = 0; c < 4; ++c) { s_extside[k][bit][c] = o[c]; s_extside[k][bit ^ 1][c] = {-o[c].re, o[c].im}; }
            }
          });
        } break;
        case T_VVV: case T_AMP_VVV: {
          const bool is_amp = tk.type() == T_AMP_VVV;
          for_items<CFG>(a, tk, nlane, i0, raw0, [&](uint32_t i, uint4 raw) {
            const uint32_t e = i & (E - 1);
            const uint32_t mA = MG_U5(raw) & 0xff, mB = MG_U5(raw) >> 8;
            Cx<T> X[4], Y[4];
            load_wf<STRIDE>(wf, MG_U0(raw) * E + e, X);
            load_wf<STRIDE>(wf, MG_U1(raw) * E + e, Y);
            const T* ma = mom + (size_t)mA * MOMSTRIDE * E + e; const T* mb = mom + (size_t)mB * MOMSTRIDE * E + e;
            T d[4], ka2[4], kb2[4];
#pragma unroll
            for (int c = 0; c < 4; ++c) { const T kA = ma[c * E], kB = mb[c * E]; d[c] = kA - kB; ka2[c] = kA + 2 * kB; kb2[c] = 2 * kA + kB; }
            const T f = mom[(size_t)(mA | mB) * MOMSTRIDE * E + 4 * E + e];
            const Cx<T> xy = mdot(X, Y), ax = rdot(ka2, X), by = rdot(kb2, Y);
            Cx<T> J[4];
#pragma unroll
            for (int c = 0; c < 4; ++c) {
              Cx<T> v = cscale(d[c], xy); cfma(v, ax, Y[c]); cfma(v, cscale((T)-1, by), X[c]);
              J[c] = {-f * v.re, -f * v.im};                     // (-i)(-i / K^2) * v: the current carries the phase of its colour factor
            }
            if (!is_amp) {
              store_wf<STRIDE>(wf, MG_U4(raw) * E + e, J);
            } else {
              // close the vertex current with the four (t, t~) variants of W0 = i ubar gamma^mu v
              const uint32_t col = MG_U6(raw), l0 = (MG_U4(raw) << CFG::LOGE) + e;
              // all four results first, then the stores: the loads of the next W do not wait behind a store
              Cx<T> v[4];
#pragma unroll
              for (int tt = 0; tt < 4; ++tt) { Cx<T> W[4]; load_wf<STRIDE>(wf, (MG_U2(raw) + tt) * E + e, W); v[tt] = mdot(J, W); }
#pragma unroll
              for (int tt = 0; tt < 4; ++tt) amp2[col * NL + l0 + ((((tt >> 1) << a.pos_t) | ((tt & 1) << a.pos_tb)) << CFG::LOGE)] = v[tt];
            }
          });
        } break;
        case T_VVVF: {
          // fused tree current (emitter/program.py fuse_quartic): the three-gluon vertex of the two children's currents plus, for
          // every composite child c = (x, y), the four-gluon structure merged into this tree, sign * ((x.z) y - (y.z) x) / K^2 with
          // z the other child's current.  u0, u1: children; u2, u3 / u6, u7: (x, y) of the first / second child; u5 = mA | mB << 5 |
          // flags << 10 (per composite child: present, negative).  PAPER.md:130-132 (VVV1 and VVVV routines in one item).
          for_items<CFG>(a, tk, nlane, i0, raw0, [&](uint32_t i, uint4 raw) {
            const uint32_t e = i & (E - 1);
            const uint32_t u5 = MG_U5(raw), mA = u5 & 31u, mB = (u5 >> 5) & 31u, fl = u5 >> 10;
            Cx<T> X[4], Y[4];
            load_wf<STRIDE>(wf, MG_U0(raw) * E + e, X);
            load_wf<STRIDE>(wf, MG_U1(raw) * E + e, Y);
            const T* ma = mom + (size_t)mA * MOMSTRIDE * E + e; const T* mb = mom + (size_t)mB * MOMSTRIDE * E + e;
            T d[4], ka2[4], kb2[4];
#pragma unroll
            for (int c = 0; c < 4; ++c) { const T kA = ma[c * E], kB = mb[c * E]; d[c] = kA - kB; ka2[c] = kA + 2 * kB; kb2[c] = 2 * kA + kB; }
            const T f = mom[(size_t)(mA | mB) * MOMSTRIDE * E + 4 * E + e];
            const Cx<T> xy = mdot(X, Y), ax = rdot(ka2, X), by = rdot(kb2, Y);
            Cx<T> J[4];
#pragma unroll
            for (int c = 0; c < 4; ++c) {
              Cx<T> v = cscale(d[c], xy); cfma(v, ax, Y[c]); cfma(v, cscale((T)-1, by), X[c]);
              J[c] = {-f * v.re, -f * v.im};
            }
            if (fl & 1u) {
              Cx<T> P[4], Q[4];
              load_wf<STRIDE>(wf, MG_U2(raw) * E + e, P);
              load_wf<STRIDE>(wf, MG_U3(raw) * E + e, Q);
              const Cx<T> c1 = mdot(P, Y), c2 = mdot(Q, Y);
              const T sf = (fl & 2u) ? -f : f;
#pragma unroll
              for (int c = 0; c < 4; ++c) { Cx<T> v = cmul(c1, Q[c]); cfma(v, cscale((T)-1, c2), P[c]); J[c].re = fma(sf, v.re, J[c].re); J[c].im = fma(sf, v.im, J[c].im); }
            }
            if (fl & 4u) {
              Cx<T> P[4], Q[4];
              load_wf<STRIDE>(wf, MG_U6(raw) * E + e, P);
              load_wf<STRIDE>(wf, MG_U7(raw) * E + e, Q);
              const Cx<T> c1 = mdot(P, X), c2 = mdot(Q, X);
              const T sf = (fl & 8u) ? -f : f;
#pragma unroll
              for (int c = 0; c < 4; ++c) { Cx<T> v = cmul(c1, Q[c]); cfma(v, cscale((T)-1, c2), P[c]); J[c].re = fma(sf, v.re, J[c].re); J[c].im = fma(sf, v.im, J[c].im); }
            }
            store_wf<STRIDE>(wf, MG_U4(raw) * E + e, J);
          });
        } break;
        case T_VVVV: case T_AMP_VVVV: {
          const bool is_amp = tk.type() == T_AMP_VVVV;
          const int s = tk.aux() & 3;
          const bool accumulate = (tk.aux() & 4) != 0;   // merged scheme: add (with sign) into the nested three-gluon tree's current
          for_items<CFG>(a, tk, nlane, i0, raw0, [&](uint32_t i, uint4 raw) {
            const uint32_t e = i & (E - 1);
            Cx<T> X[4], Y[4], Z[4];
            load_wf<STRIDE>(wf, MG_U0(raw) * E + e, X);
            load_wf<STRIDE>(wf, MG_U1(raw) * E + e, Y);
            load_wf<STRIDE>(wf, MG_U2(raw) * E + e, Z);
            const T f = mom[(size_t)(MG_U5(raw) & 0xff) * MOMSTRIDE * E + 4 * E + e];    // (-i)^2 (-i/K^2)(-i) = +1/K^2 (phase convention of VVV); mask = whole label set
            // L_0 = (X.Z) Y - (Y.Z) X ; L_1 = (X.Y) Z - (Y.Z) X ; L_2 = (X.Y) Z - (X.Z) Y
            Cx<T> c1, c2, V1[4], V2[4];
            if (s == 0) { c1 = mdot(X, Z); c2 = mdot(Y, Z); }
            else if (s == 1) { c1 = mdot(X, Y); c2 = mdot(Y, Z); }
            else { c1 = mdot(X, Y); c2 = mdot(X, Z); }
#pragma unroll
            for (int c = 0; c < 4; ++c) { V1[c] = s == 0 ? Y[c] : Z[c]; V2[c] = s == 2 ? Y[c] : X[c]; }
            Cx<T> J[4];
#pragma unroll
            for (int c = 0; c < 4; ++c) { Cx<T> v = cmul(c1, V1[c]); cfma(v, cscale((T)-1, c2), V2[c]); J[c] = cscale(f, v); }
            if (!is_amp) {
              const uint32_t so = MG_U4(raw) * E + e;
              if (accumulate) {
                const T sg = MG_U7(raw) ? (T)-1 : (T)1;
                Cx<T> O[4]; load_wf<STRIDE>(wf, so, O);
#pragma unroll
                for (int c = 0; c < 4; ++c) { O[c].re = fma(sg, J[c].re, O[c].re); O[c].im = fma(sg, J[c].im, O[c].im); }
                store_wf<STRIDE>(wf, so, O);
              } else {
                store_wf<STRIDE>(wf, so, J);
              }
            } else {
              const uint32_t col = MG_U6(raw), l0 = (MG_U4(raw) << CFG::LOGE) + e;
              const T sg = MG_U7(raw) ? (T)-1 : (T)1;
#pragma unroll
              for (int tt = 0; tt < 4; ++tt) {
                Cx<T> W[4]; load_wf<STRIDE>(wf, (MG_U3(raw) + tt) * E + e, W);
                const Cx<T> v = mdot(J, W);
                const uint32_t l = l0 + ((((tt >> 1) << a.pos_t) | ((tt & 1) << a.pos_tb)) << CFG::LOGE);
                if (accumulate) {      // folded top level: add into the column of the cubic tree with the same colour factor
                  Cx<T> o = amp2[col * NL + l];
                  o.re = fma(sg, v.re, o.re); o.im = fma(sg, v.im, o.im);
                  amp2[col * NL + l] = o;
                } else {
                  amp2[col * NL + l] = v;
                }
              }
            }
          });
        } break;
        case T_FFV: {
          for_items<CFG>(a, tk, nlane, i0, raw0, [&](uint32_t i, uint4 raw) {
            const uint32_t e = i & (E - 1);
            Cx<T> A[4], J[4], r[4], s[4];
            load_wf<STRIDE>(wf, MG_U0(raw) * E + e, A);
            load_wf<STRIDE>(wf, MG_U1(raw) * E + e, J);
            const T* mq = mom + (size_t)(MG_U5(raw) & 0xff) * MOMSTRIDE * E + e;
            const T q[4] = {mq[8 * E], mq[9 * E], mq[10 * E], mq[11 * E]};
            const Cx<T> nd = {-mq[5 * E], -mq[6 * E]};                // (i)(i) / (D + i m Gamma)
            if (CFG::DY && MG_U7(raw)) { Cx<T> J2[4]; load_wf<STRIDE>(wf, (MG_U1(raw) + MG_U7(raw)) * E + e, J2); row_slash2(A, J, J2, r); }
            else row_slash(A, J, r);
            row_slash_real_m(r, q, mt, s);
#pragma unroll
            for (int c = 0; c < 4; ++c) s[c] = cmul(nd, s[c]);
            store_wf<STRIDE>(wf, MG_U4(raw) * E + e, s);
          });
        } break;
        case T_FFVR: {
          // right chain (column spinor grown from v(t~)): S(q) slash(J) c with q = p_t - K[mask], mask = complement of the
          // chain's label set (the propagator between the closing block's side and this block)
          for_items<CFG>(a, tk, nlane, i0, raw0, [&](uint32_t i, uint4 raw) {
            const uint32_t e = i & (E - 1);
            Cx<T> C[4], J[4], r[4], s[4];
            load_wf<STRIDE>(wf, MG_U0(raw) * E + e, C);
            load_wf<STRIDE>(wf, MG_U1(raw) * E + e, J);
            const T* mq = mom + (size_t)(MG_U5(raw) & 0xff) * MOMSTRIDE * E + e;
            const T q[4] = {mq[8 * E], mq[9 * E], mq[10 * E], mq[11 * E]};
            const Cx<T> nd = {-mq[5 * E], -mq[6 * E]};                // (i)(i) / (D + i m Gamma)
            if (CFG::DY && MG_U7(raw)) { Cx<T> J2[4]; load_wf<STRIDE>(wf, (MG_U1(raw) + MG_U7(raw)) * E + e, J2); slash_col2(J, J2, C, r); }
            else slash_col(J, C, r);
            slash_real_m_col(q, mt, r, s);
#pragma unroll
            for (int c = 0; c < 4; ++c) s[c] = cmul(nd, s[c]);
            store_wf<STRIDE>(wf, MG_U4(raw) * E + e, s);
          });
        } break;
        case T_WCUR: {
          for_items<CFG>(a, tk, nlane, i0, raw0, [&](uint32_t i, uint4 raw) {
            const uint32_t e = i & (E - 1);
            Cx<T> A[4], V[4], W[4];
            load_wf<STRIDE>(wf, MG_U0(raw) * E + e, A);
            load_wf<STRIDE>(wf, MG_U1(raw) * E + e, V);
            wcurrent(A, V, W);
            store_wf<STRIDE>(wf, MG_U4(raw) * E + e, W);
          });
        } break;
        case T_COMB: {
          // colour-ordered current = signed sum of up to six tree currents of the same label set and helicities
          // (emitter/diagrams.py ordered_basis): operand slots u0..u3, u5, u6; u7 = count | signs << 3
          for_items<CFG>(a, tk, nlane, i0, raw0, [&](uint32_t i, uint4 raw) {
            const uint32_t e = i & (E - 1);
            const uint32_t n = MG_U7(raw) & 7u, sg = MG_U7(raw) >> 3;
            const uint32_t slot[6] = {MG_U0(raw), MG_U1(raw), MG_U2(raw), MG_U3(raw), MG_U5(raw), MG_U6(raw)};
            Cx<T> O[4];
#pragma unroll
            for (int c = 0; c < 4; ++c) O[c] = {(T)0, (T)0};
            // (an ordering of k gluons receives Catalan(k - 1) trees: 2 for k = 3, 5 for k = 4; k <= n_g - 1)
            constexpr int NMAX = CFG::NG <= 4 ? 2 : CFG::NG == 5 ? 5 : 6;
#pragma unroll
            for (int q = 0; q < NMAX; ++q) {
              if (q < (int)n) {
                Cx<T> X[4]; load_wf<STRIDE>(wf, slot[q] * E + e, X);
                const uint32_t sb = ((sg >> q) & 1u) << 31;
#pragma unroll
                for (int c = 0; c < 4; ++c) { O[c].re += flipsign(X[c].re, sb); O[c].im += flipsign(X[c].im, sb); }
              }
            }
            store_wf<STRIDE>(wf, MG_U4(raw) * E + e, O);
          });
        } break;
        case T_AMP_DOT: {
          // one gluon current J against the four (t, t~) variants of the chain's W current
          for_items<CFG>(a, tk, nlane, i0, raw0, [&](uint32_t i, uint4 raw) {
            const uint32_t e = i & (E - 1);
            const uint32_t pt = MG_U5(raw) & 0xff, ptb = MG_U5(raw) >> 8;
            Cx<T> J[4];
            load_wf<STRIDE>(wf, MG_U1(raw) * E + e, J);
            const uint32_t col = MG_U6(raw), l0 = (MG_U4(raw) << CFG::LOGE) + e;
            Cx<T> v[4];
#pragma unroll
            for (int tt = 0; tt < 4; ++tt) {
              Cx<T> W[4];
              load_wf<STRIDE>(wf, (MG_U0(raw) + ((tt >> 1) << pt) + ((tt & 1) << ptb)) * E + e, W);
              v[tt] = mdot(W, J);
            }
#pragma unroll
            for (int tt = 0; tt < 4; ++tt) amp2[col * NL + l0 + ((((tt >> 1) << a.pos_t) | ((tt & 1) << a.pos_tb)) << CFG::LOGE)] = v[tt];
          });
        } break;
        case T_AMP_FFV: {
          // the four (t, t~) variants of L(t) slash(J) R(t~): both left-chain rows times slash(J) are kept in registers, each
          // right-chain column (v itself for an empty right chain) is loaded once -- 20 loads for 4 amplitudes
          const uint32_t nhg = 1u << (tk.aux() & 3);      // helicity assignments of the blocked right-chain gluons per item
          for_items<CFG>(a, tk, nlane, i0, raw0, [&](uint32_t i, uint4 raw) {
            const uint32_t e = i & (E - 1);
            // u5: bit positions as nibbles: t~ in the right chain's variant index | blocked gluon there << 4 | t in the left
            // chain's << 8 | blocked gluon in the helicity combination << 12; u7: the same two for a second blocked gluon.
            // aux = number of gluons that enter only through the right chain and whose helicities the item runs over
            // (8 or 16 amplitudes from the same two rows L(t) slash(J))
            const uint32_t u5 = MG_U5(raw), sh_tb = u5 & 15u, sh_g = (u5 >> 4) & 15u, sh_t = (u5 >> 8) & 15u, lsh_g = u5 >> 12;
            Cx<T> J[4], r0[4], r1[4];
            load_wf<STRIDE>(wf, MG_U1(raw) * E + e, J);
            const uint32_t chir = CFG::DY ? MG_U7(raw) >> 8 : 0u;         // Drell-Yan: offset of the current's right-chiral partner
            if (chir) {
              Cx<T> J2[4], A[4];
              load_wf<STRIDE>(wf, (MG_U1(raw) + chir) * E + e, J2);
              load_wf<STRIDE>(wf, MG_U0(raw) * E + e, A); row_slash2(A, J, J2, r0);
              load_wf<STRIDE>(wf, (MG_U0(raw) + (1u << sh_t)) * E + e, A); row_slash2(A, J, J2, r1);
            } else {
            { Cx<T> A[4]; load_wf<STRIDE>(wf, MG_U0(raw) * E + e, A); row_slash(A, J, r0); }
            { Cx<T> A[4]; load_wf<STRIDE>(wf, (MG_U0(raw) + (1u << sh_t)) * E + e, A); row_slash(A, J, r1); }
            }
            const uint32_t col = MG_U6(raw), l00 = (MG_U4(raw) << CFG::LOGE) + e;
            const uint32_t sh_g1 = MG_U7(raw) & 15u, lsh_g1 = (MG_U7(raw) >> 4) & 15u;
            for (uint32_t hg = 0; hg < nhg; ++hg) {
              const uint32_t rbase = MG_U2(raw) + ((hg & 1u) << sh_g) + ((hg >> 1) << sh_g1);
              const uint32_t l0 = l00 + ((((hg & 1u) << lsh_g) + ((hg >> 1) << lsh_g1)) << CFG::LOGE);
              Cx<T> v0[2], v1[2];
#pragma unroll
              for (int tb = 0; tb < 2; ++tb) {
                Cx<T> V[4]; load_wf<STRIDE>(wf, (rbase + (tb << sh_tb)) * E + e, V);
                v0[tb] = cmul(r0[0], V[0]); cfma(v0[tb], r0[1], V[1]); cfma(v0[tb], r0[2], V[2]); cfma(v0[tb], r0[3], V[3]);
                v1[tb] = cmul(r1[0], V[0]); cfma(v1[tb], r1[1], V[1]); cfma(v1[tb], r1[2], V[2]); cfma(v1[tb], r1[3], V[3]);
              }
#pragma unroll
              for (int tb = 0; tb < 2; ++tb) {
                const uint32_t l = l0 + ((tb << a.pos_tb) << CFG::LOGE);
                amp2[col * NL + l] = {-v0[tb].im, v0[tb].re};   // i * v
                amp2[col * NL + l + ((1u << a.pos_t) << CFG::LOGE)] = {-v1[tb].im, v1[tb].re};
              }
            }
          });
        } break;
        case T_QSUM: {
          // Colour-ordered quark line (emitter/program.py _chains_bg): row sum A = sum_j r_j A_j slash(J_j) over up to four
          // (row spinor, ordered current) pairs, r_j = +-1.  aux = 0: times the quark propagator S(p_t - K[mask]) -> the quark
          // current of the ordered gluon prefix.  aux = 1: closing sum of a colour flow for both t~ helicities,
          //   jamp[flow] += i (A . R1(t~) + B . v(t~)),  B = a second row sum of up to three pairs.
          // 48-byte entries: word 0 = A0 J0 A1 J1 | result slot or helicity combination | flags | flow or subset | bit of t~ in R1,
          // word 1 = A2 J2 A3 J3 | R1 | v, word 2 = the pairs of B; flags = terms A | terms B << 3 | signs A << 6 | signs B << 10.
          const bool closing = (tk.aux() & 1u) != 0;
          const uint4* tbl = reinterpret_cast<const uint4*>(a.idx) + tk.tbl_off();
          uint32_t i = i0;
          uint4 w0 = raw0, w1 = make_uint4(0, 0, 0, 0), w2 = w1;
          if (i < nlane) { w1 = __ldg(tbl + 3 * (i >> CFG::LOGE) + 1); if (closing) w2 = __ldg(tbl + 3 * (i >> CFG::LOGE) + 2); }
          while (i < nlane) {
            const uint32_t in = i + 32;
            uint4 n0 = w0, n1 = w1, n2 = w2;
            if (in < nlane) {
              const uint4* q = tbl + 3 * (in >> CFG::LOGE);
              n0 = __ldg(q); n1 = __ldg(q + 1);
              if (closing) n2 = __ldg(q + 2);
            }
            const uint32_t e = i & (E - 1);
            const uint32_t fl = MG_U5(w0), nA = fl & 7u, sgA = (fl >> 6) & 15u, sgB = (fl >> 10) & 7u;
            const uint32_t sa[4] = {MG_U0(w0), MG_U2(w0), MG_U0(w1), MG_U2(w1)}, ja[4] = {MG_U1(w0), MG_U3(w0), MG_U1(w1), MG_U3(w1)};
            if (!closing) {
              Cx<T> rA[4];
#pragma unroll
              for (int c = 0; c < 4; ++c) rA[c] = {(T)0, (T)0};
#pragma unroll
              for (int q = 0; q < 4; ++q) {
                if (q < CFG::NG - 1 && q < (int)nA) {      // at most n_g - 1 terms: the code of the others is not generated
                  Cx<T> A[4], J[4];
                  load_wf<STRIDE>(wf, sa[q] * E + e, A);
                  load_wf<STRIDE>(wf, ja[q] * E + e, J);
                  row_slash_acc(A, J, (sgA >> q) << 31, rA);
                }
              }
              const T* mq = mom + (size_t)(MG_U6(w0) & 0xff) * MOMSTRIDE * E + e;
              const T q[4] = {mq[8 * E], mq[9 * E], mq[10 * E], mq[11 * E]};
              const Cx<T> nd = {-mq[5 * E], -mq[6 * E]};                // (i)(i) / (D + i m Gamma)
              Cx<T> s[4];
              row_slash_real_m(rA, q, mt, s);
#pragma unroll
              for (int c = 0; c < 4; ++c) s[c] = cmul(nd, s[c]);
              store_wf<STRIDE>(wf, MG_U4(w0) * E + e, s);
            } else {
              // Term j of the second row sum uses the same row spinor Q[sigma_1..sigma_j] as term j of the first one (j >= 1), so it is
              // loaded once: 60 instead of 72 128-bit loads per item in a phase that is bound by the shared-memory pipe.
              const uint32_t jb[3] = {MG_U1(w2), MG_U3(w2), MG_U5(w2)};
              Cx<T> rA[4], rB[4];
              {
                Cx<T> A[4], J[4];
                load_wf<STRIDE>(wf, sa[0] * E + e, A);
                load_wf<STRIDE>(wf, ja[0] * E + e, J);
#pragma unroll
                for (int c = 0; c < 4; ++c) J[c] = {flipsign(J[c].re, sgA << 31), flipsign(J[c].im, sgA << 31)};
                row_slash(A, J, rA);
              }
#pragma unroll
              for (int c = 0; c < 4; ++c) rB[c] = {(T)0, (T)0};
#pragma unroll
              for (int q = 1; q < 4; ++q) {
                if (q < CFG::NG - 1 && q < (int)nA) {      // at most n_g - 1 terms: the code of the others is not generated
                  Cx<T> A[4], J[4];
                  load_wf<STRIDE>(wf, sa[q] * E + e, A);
                  load_wf<STRIDE>(wf, ja[q] * E + e, J);
                  row_slash_acc(A, J, (sgA >> q) << 31, rA);
                  load_wf<STRIDE>(wf, jb[q - 1] * E + e, J);
                  row_slash_acc(A, J, (sgB >> (q - 1)) << 31, rB);
                }
              }
              const uint32_t flow = MG_U6(w0), sh_tb = MG_U7(w0);
              Cx<T> v[2];
#pragma unroll
              for (int tb = 0; tb < 2; ++tb) {
                Cx<T> R[4], V[4];
                load_wf<STRIDE>(wf, (MG_U4(w1) + ((uint32_t)tb << sh_tb)) * E + e, R);
                load_wf<STRIDE>(wf, (MG_U5(w1) + tb) * E + e, V);
                v[tb] = cmul(rA[0], R[0]); cfma(v[tb], rA[1], R[1]); cfma(v[tb], rA[2], R[2]); cfma(v[tb], rA[3], R[3]);
                cfma(v[tb], rB[0], V[0]); cfma(v[tb], rB[1], V[1]); cfma(v[tb], rB[2], V[2]); cfma(v[tb], rB[3], V[3]);
              }
#pragma unroll
              for (int tb = 0; tb < 2; ++tb) {
                const uint32_t l = ((MG_U4(w0) | ((uint32_t)tb << a.pos_tb)) << CFG::LOGE) + e;
                Cx<T>* jp = jamp2 + flow * NL + (l ^ CFG::swz(flow));
                Cx<T> j = *jp;
                j.re -= v[tb].im; j.im += v[tb].re;          // += i * v
                *jp = j;
              }
            }
            i = in; w0 = n0; w1 = n1; w2 = n2;
          }
        } break;
        default: break;
      }
    }
    tk = tk1; i0 = i0n; nlane = nlanen; raw0 = raw0n;
  }
  __syncthreads();

  if constexpr (CHAN) {
    // ---- multichannel: sum the lanes' channel sums over the good inner helicities, per event -----------------------------
    if (tid < NL) {
      const int l = (int)tid, c = l >> CFG::LOGE;
      const bool ok = a.good[a.hout[outer] + a.hin[c]] != 0;
      double num = ok ? chansum[l] : 0.0, den = ok ? chansum[NL + l] : 0.0;
#pragma unroll
      for (int off = 16; off >= E; off >>= 1) { num += __shfl_xor_sync(0xffffffffu, num, off); den += __shfl_xor_sync(0xffffffffu, den, off); }
      if ((int)lane < E) {
        const long long ev = ev0 + lane;
        const double g2 = gsE[lane] * gsE[lane];
        double gp = 1;
#pragma unroll
        for (int k = 0; k < CFG::NGLUON; ++k) gp *= g2;
        if (ev < a.nevt) {
          double* o = a.chanpart + ((ev * CFG::NOUTER + outer) * (NL / 32) + warp) * 2;
          o[0] = num * gp; o[1] = den * gp;
        }
      }
    }
  } else {
  // ---- colour-flow weights: sum over the inner helicities of |J_{h,c}|^2 --------------------------------------------
  if constexpr (E == 1 && NL == 32 && NT >= 4 * NCOLOR) {
    // thread = (flow, quarter of the 32 helicity lanes); the 8 lanes of a quarter-warp (2 flows x 4 quarters) read 8 distinct
    // 16-byte bank groups per step.  With the outer-helicity passes of an event back to back in this CTA (PER_TILE) the weight
    // stays in a register across the passes and goes to global memory once per event.
    const int s = (int)(tid >> 2), part = (int)(tid & 3u);
    double v = 0;
    if (s < NCOLOR) {
#pragma unroll
      for (int k = 0; k < 8; ++k) {
        const Cx<T> js = jamp2[s * 32 + part * 8 + ((k + s + 2 * part) & 7)];
        const double re = (double)js.re, im = (double)js.im;
        v = fma(re, re, v); v = fma(im, im, v);
      }
    }
    v += __shfl_xor_sync(0xffffffffu, v, 1); v += __shfl_xor_sync(0xffffffffu, v, 2);
    wacc += v;
    if (!PER_TILE || pass == CFG::NOUTER - 1) {
      if (part == 0 && s < NCOLOR && ev0 < a.nevt) {
        const double g2 = gsE[0] * gsE[0];
        double gp = 1;
#pragma unroll
        for (int k = 0; k < CFG::NGLUON; ++k) gp *= g2;
        a.wpart[(ev0 * (PER_TILE ? 1 : CFG::NOUTER) + (PER_TILE ? 0 : outer)) * NCOLOR + (CFG::DMMA ? (int)a.flowslot[s] : s)] = wacc * gp;
      }
      wacc = 0;
    }
  } else {
    constexpr int nwarp = NT >> 5;
    for (int s = warp; s < NCOLOR; s += nwarp) {
      double v = 0;
      for (int l = lane; l < NL; l += 32) {
        const Cx<T> js = jamp2[s * NL + l];
        const double re = (double)js.re, im = (double)js.im;
        v += re * re + im * im;
      }
#pragma unroll
      for (int off = 16; off >= E; off >>= 1) v += __shfl_xor_sync(0xffffffffu, v, off);
      if ((int)lane < E) {
        const long long ev = ev0 + lane;
        const double g2 = gsE[lane] * gsE[lane];
        double gp = 1;
#pragma unroll
        for (int k = 0; k < CFG::NGLUON; ++k) gp *= g2;
        if (ev < a.nevt) a.wpart[(ev * CFG::NOUTER + outer) * NCOLOR + (CFG::DMMA ? (int)a.flowslot[s] : s)] = v * gp;
      }
    }
  }
  // ---- colour sum |M_h|^2 = J^dagger C J per (inner helicity, event) lane; C = numerators / colden ---------------
  if constexpr (CFG::DMMA && std::is_same<T, double>::value && std::is_same<TC, double>::value) {
    // FP64 tensor cores ("a single matrix multiplication"; measured on B200 by mg_measure_fp64_pipes: DMMA fed
    // from this shared-memory layout runs at 36.9 TFLOP/s against 23.7 for the DFMA form, on the same pipe).
    // X[row = 2 * lane + part][flow] (64 x NCOLOR) is the jamp tile; Y = X C' with C' = C on the diagonal 8 x 8 blocks, 2 C
    // above, 0 below (C symmetric); |M|^2[lane] = sum over both parts and all flows of Y o X.  A warp owns MTW m-tiles of 8
    // rows and the n-blocks of one group; B fragments stream from global memory (L2), once per block pair for all its m-tiles.
    // J+- = J_sigma +- J_reversed in place (slots k and HALF + k; the flow weights above were taken from the J's)
    __syncthreads();
    for (int i = tid; i < CFG::HALF * 32; i += NT) {
      const uint32_t k = (uint32_t)i >> 5, l = (uint32_t)i & 31u;
      Cx<T>* pa = jamp2 + k * 32 + (l ^ CFG::swz(k));
      Cx<T>* pb = jamp2 + (CFG::HALF + k) * 32 + (l ^ CFG::swz(CFG::HALF + k));
      const Cx<T> x = *pa, y = *pb;
      *pa = {x.re + y.re, x.im + y.im}; *pb = {x.re - y.re, x.im - y.im};
    }
    __syncthreads();
    constexpr int NB = NCOLOR / 8, NWARP = NT / 32;
    constexpr int MSPLIT = NWARP >= 16 ? 2 : (NWARP >= 4 ? 4 : NWARP), NSPLIT = NWARP / MSPLIT, MTW = 8 / MSPLIT;
    static_assert(MSPLIT * NSPLIT == NWARP && MTW * MSPLIT == 8, "warps must tile the 8 m-tiles");
    const int mg = warp % MSPLIT, ng = warp / MSPLIT;
    const double* X = reinterpret_cast<const double*>(jamp);
    const int r0 = mg * MTW * 8 + (int)(lane >> 2), kq = (int)(lane & 3);
    double part[MTW];
#pragma unroll
    for (int m = 0; m < MTW; ++m) part[m] = 0.0;
    for (int nb = 0; nb < NB; ++nb) {
      if ((nb < NSPLIT ? nb : (NB - 1 - nb) % NSPLIT) != ng) continue;
      double acc[MTW][2];
#pragma unroll
      for (int m = 0; m < MTW; ++m) { acc[m][0] = 0.0; acc[m][1] = 0.0; }
      const int kb0 = CFG::kb_lo(nb);
      const double* bf = a.colfrag + ((size_t)CFG::frag_off(nb) * 2) * 32 + lane;
      double b0 = __ldg(bf), b1 = __ldg(bf + 32);
      for (int kb = kb0; kb <= nb; ++kb) {
        double n0 = b0, n1 = b1;
        if (kb < nb) { n0 = __ldg(bf + (kb - kb0 + 1) * 64); n1 = __ldg(bf + (kb - kb0 + 1) * 64 + 32); }
#pragma unroll
        for (int ks = 0; ks < 2; ++ks) {
          const uint32_t k = (uint32_t)(kb * 8 + ks * 4 + kq);
          const double* xk = X + k * 64;
          const uint32_t sw = CFG::swz(k) << 1;
#pragma unroll
          for (int m = 0; m < MTW; ++m) mg_dmma_f64(acc[m][0], acc[m][1], xk[(uint32_t)(r0 + m * 8) ^ sw], ks ? b1 : b0);
        }
        b0 = n0; b1 = n1;
      }
      // Y o X on the accumulator layout: thread holds Y[row = lane / 4][columns 2 * (lane % 4), + 1] of every m-tile
      const uint32_t t0 = (uint32_t)(nb * 8 + 2 * kq);
#pragma unroll
      for (int m = 0; m < MTW; ++m) {
        const uint32_t r = (uint32_t)(r0 + m * 8);
        part[m] = fma(acc[m][0], X[t0 * 64 + (r ^ (CFG::swz(t0) << 1))], part[m]);
        part[m] = fma(acc[m][1], X[(t0 + 1) * 64 + (r ^ (CFG::swz(t0 + 1) << 1))], part[m]);
      }
    }
    // reduce over the four column pairs of a row (lane % 4) and over the (re, im) rows of a helicity lane (lane / 4 parity)
#pragma unroll
    for (int m = 0; m < MTW; ++m) {
      double v = part[m];
      v += __shfl_xor_sync(0xffffffffu, v, 1); v += __shfl_xor_sync(0xffffffffu, v, 2); v += __shfl_xor_sync(0xffffffffu, v, 4);
      if ((lane & 7) == 0) red[ng * 32 + (mg * MTW + m) * 4 + (lane >> 3)] = v;
    }
    __syncthreads();
    if (tid < 32) {
      double sum = 0;
#pragma unroll
      for (int g = 0; g < NSPLIT; ++g) sum += red[g * 32 + tid];
      const long long ev = ev0;
      if (ev < a.nevt) {
        const double g2 = gsE[0] * gsE[0];
        double gp = 1;
#pragma unroll
        for (int k = 0; k < CFG::NGLUON; ++k) gp *= g2;
        a.mh2[ev * CFG::NCOMB + a.hout[outer] + a.hin[tid]] = sum * a.inv_colden * gp;
      }
    }
  } else
  // thread (g, l): RPT rows of C (row group g) against all NCOLOR columns; C blocked as [g][column][RPT]
  {
    constexpr int G = CFG::G, RPT = CFG::RPT;
    constexpr int GU = (NCOLOR + RPT - 1) / RPT;                    // row groups that hold rows
    constexpr int CBYTES = GU * NCOLOR * RPT * (int)sizeof(TC);
    constexpr int CWORDS = (CBYTES + 15) / 16;                      // (the device array is padded to whole 16-byte words)
    static_assert((size_t)CWORDS * 16 <= (8 * (size_t)STRIDE + (size_t)(CFG::NCOL + 1) * 2 * NL) * sizeof(T),
                  "colour matrix must fit in the dead wavefunction / amplitude-buffer block");
    // the wavefunction file is dead now: stage the blocked colour matrix in it (one coalesced pass), then broadcast-read it
    TC* Cs = reinterpret_cast<TC*>(wf);
    {
      const uint4* src = reinterpret_cast<const uint4*>(a.colmat);
      uint4* dst = reinterpret_cast<uint4*>(Cs);
      for (int i = tid; i < CWORDS; i += NT) dst[i] = __ldg(src + i);
    }
    __syncthreads();
    // C is symmetric: only the upper block triangle is used (the staged matrix holds C on the diagonal blocks, 2C above,
    // 0 below).  The (row group g, column t >= g * RPT) iteration space is cut into G equal chunks, one per worker
    // (= NL threads sharing tid / NL); a chunk spans at most a few row groups.
    const int l = tid % NL, wk = tid / NL;
    constexpr int NIT = GU * NCOLOR - RPT * (GU * (GU - 1) / 2);     // sum over g of (NCOLOR - g * RPT)
    constexpr int CHUNK = (NIT + G - 1) / G;
    TC part = 0;
    {
      int it = wk * CHUNK, left = NIT - it < CHUNK ? NIT - it : CHUNK;
      int g = 0;
      while (g < GU && it >= NCOLOR - g * RPT) { it -= NCOLOR - g * RPT; ++g; }
      while (left > 0 && g < GU) {
        const int t_lo = g * RPT + it;
        const int n = NCOLOR - t_lo < left ? NCOLOR - t_lo : left;
        const TC* Cg = Cs + (size_t)g * NCOLOR * RPT;
        TC tx[RPT], ty[RPT];
#pragma unroll
        for (int r = 0; r < RPT; ++r) { tx[r] = 0; ty[r] = 0; }
#pragma unroll 4
        for (int t = t_lo; t < t_lo + n; ++t) {
          const Cx<T> jt = jamp2[t * NL + (l ^ (int)CFG::swz(t))];
          const TC x = (TC)jt.re, y = (TC)jt.im;
#pragma unroll
          for (int r = 0; r < RPT; ++r) { const TC c = Cg[t * RPT + r]; tx[r] = fma(c, x, tx[r]); ty[r] = fma(c, y, ty[r]); }
        }
#pragma unroll
        for (int r = 0; r < RPT; ++r) {
          const int s2 = g * RPT + r;
          if (s2 < NCOLOR) { const Cx<T> js = jamp2[s2 * NL + (l ^ (int)CFG::swz(s2))]; part = fma((TC)js.re, tx[r], part); part = fma((TC)js.im, ty[r], part); }
        }
        left -= n; it = 0; ++g;
      }
    }
    const int g = wk;
    red[tid] = (double)part;
    __syncthreads();
    if (g == 0) {
      double sum = 0;
#pragma unroll
      for (int gg = 0; gg < G; ++gg) sum += red[gg * NL + l];
      const int e = l & (E - 1), c = l >> CFG::LOGE;
      const long long ev = ev0 + e;
      if (ev < a.nevt) {
        const double g2 = gsE[e] * gsE[e];
        double gp = 1;
#pragma unroll
        for (int k = 0; k < CFG::NGLUON; ++k) gp *= g2;
        a.mh2[ev * CFG::NCOMB + a.hout[outer] + a.hin[c]] = sum * a.inv_colden * gp;
      }
    }
  }
  }                     // (not the multichannel program)
  __syncthreads();      // shared memory is reused by the next pass
  }
  }
}
