// mg_lib.cu -- C ABI (include/mg5b200.h) and the auxiliary kernels of the B200 matrix-element library:
// Philox4x32-10 + RAMBO sampler (a0), e+e- -> mu+mu- kernel (config 1), helicity/colour selection and store
// (a6-a8, a10), helicity filter (a9), FMA-peak microbenchmark.  The QCD wavefunction VM is in mg_vm.cuh.
// No CPU fallback: every entry point that computes launches kernels on the context's device.
#include <cmath>
#include <cstdio>
#include <cstring>
#include <new>
#include <vector>

#include "../../include/mg5b200.h"
#include "mg_vm.cuh"
#include "mg_pipes.cuh"
#include "generated/mg_programs.inc"

// =================================================================================================================
// Philox4x32-10 (Salmon et al. 2011) -- DESIGN.md "Uniforms": key = seed, counter = (event lo, event hi, block, purpose)
// =================================================================================================================
__device__ __forceinline__ void philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, uint32_t k0, uint32_t k1, uint32_t* out) {
#pragma unroll
  for (int r = 0; r < 10; ++r) {
    if (r > 0) { k0 += 0x9E3779B9u; k1 += 0xBB67AE85u; }
    uint32_t hi0 = __umulhi(0xD2511F53u, c0), lo0 = 0xD2511F53u * c0;
    uint32_t hi1 = __umulhi(0xCD9E8D57u, c2), lo1 = 0xCD9E8D57u * c2;
    uint32_t n0 = hi1 ^ c1 ^ k0, n2 = hi0 ^ c3 ^ k1;
    c0 = n0; c1 = lo1; c2 = n2; c3 = lo0;
  }
  out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}
__device__ __forceinline__ void uniforms2(unsigned long long seed, unsigned long long event, uint32_t block, uint32_t purpose, double* u) {
  uint32_t w[4];
  philox4x32_10((uint32_t)event, (uint32_t)(event >> 32), block, purpose, (uint32_t)seed, (uint32_t)(seed >> 32), w);
  unsigned long long a = ((unsigned long long)w[0] << 32) | w[1], b = ((unsigned long long)w[2] << 32) | w[3];
  const double s = 1.0 / 9007199254740992.0;
  u[0] = (double)(2 * (a >> 12) + 1) * s;
  u[1] = (double)(2 * (b >> 12) + 1) * s;
}

__device__ __forceinline__ size_t mom_index(long long ev, int npar, int leg, int c, int layout) {
  return layout == MG_LAYOUT_AOS ? (size_t)((ev * npar + leg) * 4 + c) : (size_t)((((ev >> 5) * npar + leg) * 4 + c) * 32 + (ev & 31));
}

// =================================================================================================================
// a0: RAMBO sampler, one event per thread
// =================================================================================================================
struct RamboArgs { unsigned long long seed, first; int nevt, nf, layout; double E; double mass[6]; double* p; double* w; };

__global__ void __launch_bounds__(128) mg_rambo_kernel(const RamboArgs a) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= a.nevt) return;
  const double PI = 3.14159265358979323846;
  const int nf = a.nf, npar = nf + 2;
  const double E = a.E;
  double q[6][4], Q[4] = {0, 0, 0, 0};
#pragma unroll
  for (int k = 0; k < 6; ++k) if (k < nf) {
    double r[4];
    uniforms2(a.seed, a.first + i, 2 * k, 0u, r);
    uniforms2(a.seed, a.first + i, 2 * k + 1, 0u, r + 2);
    double c = 2 * r[0] - 1, phi = 2 * PI * r[1];
    double q0 = -log(r[2] * r[3]);
    double st = sqrt(1 - c * c);
    q[k][0] = q0; q[k][1] = q0 * st * cos(phi); q[k][2] = q0 * st * sin(phi); q[k][3] = q0 * c;
    for (int m = 0; m < 4; ++m) Q[m] += q[k][m];
  }
  double M2 = Q[0] * Q[0] - Q[1] * Q[1] - Q[2] * Q[2] - Q[3] * Q[3];
  if (!(M2 > 0)) {                    // cancelled to <= 0 (near-collinear massless pair): M^2 = 2 sum_{i<j} q_i.q_j has no cancellation
    M2 = 0;
    for (int k = 0; k < 6; ++k) for (int j = k + 1; j < 6; ++j) if (j < nf)
      M2 += 2 * (q[k][0] * q[j][0] - q[k][1] * q[j][1] - q[k][2] * q[j][2] - q[k][3] * q[j][3]);
  }
  double M = sqrt(M2);
  double b[3] = {-Q[1] / M, -Q[2] / M, -Q[3] / M};
  double x = E / M, gam = Q[0] / M, aa = 1 / (1 + gam);
  double pf[6][4], e[6];
  bool massive = false; double summ = 0;
#pragma unroll
  for (int k = 0; k < 6; ++k) if (k < nf) {
    double bq = b[0] * q[k][1] + b[1] * q[k][2] + b[2] * q[k][3];
    pf[k][0] = x * (gam * q[k][0] + bq);
    for (int m = 0; m < 3; ++m) pf[k][1 + m] = x * (q[k][1 + m] + b[m] * q[k][0] + aa * bq * b[m]);
    e[k] = sqrt(pf[k][1] * pf[k][1] + pf[k][2] * pf[k][2] + pf[k][3] * pf[k][3]);
    if (a.mass[k] != 0) massive = true;
    summ += a.mass[k];
  }
  double fact = 1;
  for (int k = 2; k <= nf - 1; ++k) fact *= k;
  for (int k = 2; k <= nf - 2; ++k) fact *= k;
  double W = pow(PI / 2, (double)(nf - 1)) * pow(E, (double)(2 * nf - 4)) / fact * pow(2 * PI, (double)(4 - 3 * nf));
  if (!massive) {
#pragma unroll
    for (int k = 0; k < 6; ++k) if (k < nf) pf[k][0] = e[k];
  } else {
    double xi = sqrt(1 - (summ / E) * (summ / E));
    for (int it = 0; it < 16; ++it) {
      double f = -E, df = 0;
#pragma unroll
      for (int k = 0; k < 6; ++k) if (k < nf) {
        double en = sqrt(a.mass[k] * a.mass[k] + xi * xi * e[k] * e[k]);
        f += en; df += xi * e[k] * e[k] / en;
      }
      if (fabs(f) < 1e-15 * E) break;
      xi -= f / df;
    }
    double sumk = 0, prod = 1, sumk2 = 0;
#pragma unroll
    for (int k = 0; k < 6; ++k) if (k < nf) {
      for (int m = 1; m < 4; ++m) pf[k][m] *= xi;
      double kk = xi * e[k];
      double k0 = sqrt(a.mass[k] * a.mass[k] + kk * kk);
      pf[k][0] = k0;
      sumk += kk; prod *= kk / k0; sumk2 += kk * kk / k0;
    }
    W *= pow(sumk / E, (double)(2 * nf - 3)) * prod / sumk2 * E;
  }
  long long ev = i;
  double beam[2][4] = {{E / 2, 0, 0, E / 2}, {E / 2, 0, 0, -E / 2}};
  for (int leg = 0; leg < 2; ++leg) for (int c = 0; c < 4; ++c) a.p[mom_index(ev, npar, leg, c, a.layout)] = beam[leg][c];
#pragma unroll
  for (int k = 0; k < 6; ++k) if (k < nf) for (int c = 0; c < 4; ++c) a.p[mom_index(ev, npar, 2 + k, c, a.layout)] = pf[k][c];
  if (a.w) a.w[i] = W;
}

__global__ void mg_uniforms_kernel(unsigned long long seed, unsigned long long first, int nevt, double* rh, double* rc) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= nevt) return;
  double u[2];
  uniforms2(seed, first + i, 0u, 1u, u);
  if (rh) rh[i] = u[0];
  if (rc) rc[i] = u[1];
}

// =================================================================================================================
// config 1: e+(0) e-(1) -> mu+(2) mu-(3) via photon + Z, one event per thread
// =================================================================================================================
struct EEArgs { const double* p; int nevt, layout; double MZ, WZ, gLA, gRA, gLZ, gRZ; double* mh2; unsigned long long mask; };

// massless spinors: chi_lambda two-spinors and sqrt(2|p|)
__device__ __forceinline__ void ee_chis(const double* p, Cx<double> xp[2], Cx<double> xm[2], double& w) {
  double pp = sqrt(p[1] * p[1] + p[2] * p[2] + p[3] * p[3]);
  w = sqrt(2 * pp);
  ext_chi<double>(p, pp, +1, xp);
  ext_chi<double>(p, pp, -1, xm);
}
__device__ __forceinline__ Cx<double> cconj(Cx<double> a) { return {a.re, -a.im}; }

__global__ void __launch_bounds__(128) mg_ee_kernel(const EEArgs a) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= a.nevt) return;
  double p[4][4];
  for (int leg = 0; leg < 4; ++leg) for (int c = 0; c < 4; ++c) p[leg][c] = a.p[mom_index(i, 4, leg, c, a.layout)];
  // spinors per leg and helicity, as (column or row) 4-spinors; massless => two non-zero components
  // leg 0: incoming e+  -> vbar(p0, lam);  leg 1: incoming e- -> u(p1, lam);
  // leg 2: outgoing mu+ -> v(p2, lam);     leg 3: outgoing mu- -> ubar(p3, lam)
  Cx<double> sp[4][2][4];
  for (int leg = 0; leg < 4; ++leg) {
    Cx<double> xp[2], xm[2]; double w;
    ee_chis(p[leg], xp, xm, w);
    for (int b = 0; b < 2; ++b) {
      int lam = b ? 1 : -1;
      Cx<double> s[4] = {{0, 0}, {0, 0}, {0, 0}, {0, 0}};
      bool is_u = (leg == 1 || leg == 3);
      if (is_u) {   // u = (omega_{-lam} chi_lam ; omega_lam chi_lam), omega_- = 0
        const Cx<double>* x = lam > 0 ? xp : xm;
        int o = lam > 0 ? 2 : 0;
        s[o] = cscale(w, x[0]); s[o + 1] = cscale(w, x[1]);
      } else {      // v = (-lam omega_lam chi_{-lam} ; lam omega_{-lam} chi_{-lam})
        const Cx<double>* x = lam > 0 ? xm : xp;
        if (lam > 0) { s[0] = cscale(-w, x[0]); s[1] = cscale(-w, x[1]); } else { s[2] = cscale(-w, x[0]); s[3] = cscale(-w, x[1]); }
      }
      bool bar = (leg == 0 || leg == 3);
      if (bar) { Cx<double> t[4] = {cconj(s[2]), cconj(s[3]), cconj(s[0]), cconj(s[1])}; for (int c = 0; c < 4; ++c) s[c] = t[c]; }
      for (int c = 0; c < 4; ++c) sp[leg][b][c] = s[c];
    }
  }
  double s = 0;
  { double k[4]; for (int c = 0; c < 4; ++c) k[c] = p[0][c] + p[1][c]; s = k[0] * k[0] - k[1] * k[1] - k[2] * k[2] - k[3] * k[3]; }
  // propagator factors i / den
  Cx<double> propA = {0.0, 1.0 / s};
  double dz = s - a.MZ * a.MZ, gz = a.MZ * a.WZ, nz = dz * dz + gz * gz;
  Cx<double> propZ = {gz / nz, dz / nz};   // i / (dz + i gz) = i (dz - i gz)/nz
  for (int h = 0; h < 16; ++h) {
    double val = 0;
    if (a.mask >> h & 1) {
      int b0 = h >> 3 & 1, b1 = h >> 2 & 1, b2 = h >> 1 & 1, b3 = h & 1;
      // chiral currents: abar gamma^mu P_L b (upper components of b) and P_R (lower components)
      Cx<double> JeL[4], JeR[4], JmL[4], JmR[4];
      for (int side = 0; side < 2; ++side) {
        const Cx<double>* ab = side == 0 ? sp[0][b0] : sp[3][b3];
        const Cx<double>* bb = side == 0 ? sp[1][b1] : sp[2][b2];
        Cx<double>* L = side == 0 ? JeL : JmL; Cx<double>* R = side == 0 ? JeR : JmR;
        Cx<double> t20 = cmul(ab[2], bb[0]), t31 = cmul(ab[3], bb[1]), t21 = cmul(ab[2], bb[1]), t30 = cmul(ab[3], bb[0]);
        L[0] = cadd(t20, t31); L[1] = cscale(-1.0, cadd(t21, t30));
        Cx<double> d = csub(t21, t30); L[2] = {-d.im, d.re};           // i (a2 b1 - a3 b0)
        L[3] = cscale(-1.0, csub(t20, t31));
        Cx<double> u02 = cmul(ab[0], bb[2]), u13 = cmul(ab[1], bb[3]), u03 = cmul(ab[0], bb[3]), u12 = cmul(ab[1], bb[2]);
        R[0] = cadd(u02, u13); R[1] = cadd(u03, u12);
        Cx<double> d2 = csub(u12, u03); R[2] = {-d2.im, d2.re};        // i (-a0 b3 + a1 b2)
        R[3] = csub(u02, u13);
      }
      Cx<double> M = {0, 0};
      for (int V = 0; V < 2; ++V) {
        double gL = V ? a.gLZ : a.gLA, gR = V ? a.gRZ : a.gRA;
        Cx<double> Je[4], Jm[4];
        for (int c = 0; c < 4; ++c) { Je[c] = cadd(cscale(gL, JeL[c]), cscale(gR, JeR[c])); Jm[c] = cadd(cscale(gL, JmL[c]), cscale(gR, JmR[c])); }
        Cx<double> d = mdot(Je, Jm);       // (-i)^3 (Je.Jm) / den = i (Je.Jm) / den
        M = cadd(M, cmul(V ? propZ : propA, d));
      }
      val = M.re * M.re + M.im * M.im;
    }
    a.mh2[(size_t)i * 16 + h] = val;
  }
}

// =================================================================================================================
// a6-a8, a10: helicity sum, helicity and colour selection, store.  One event per thread.
// =================================================================================================================
struct FinArgs {
  const double* mh2; const double* wpart; const unsigned char* good; const double* rh; const double* rc;
  double* me; int* sel_hel; int* sel_col; double* wcol_out;
  int nevt, ncomb, ncolor, nouter, denom;      // wpart[nevt][nouter][ncolor] carries g_s^(2 ng) already
  // multichannel: the colour is selected among the flows the event's channel contributes to
  const int* channel;                // [ceil(nevt / 32)] 1-based channel per 32-event block, 0 = none; NULL = none
  const unsigned char* chanflows;    // [nchan][ncolor]
};

__global__ void __launch_bounds__(128) mg_finalize_kernel(const FinArgs a) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= a.nevt) return;
  const double* m = a.mh2 + (size_t)i * a.ncomb;
  double T = 0;
  for (int h = 0; h < a.ncomb; ++h) if (a.good[h]) T += m[h];
  a.me[i] = T / (double)a.denom;
  if (a.sel_hel && a.rh) {
    double r = a.rh[i] * T, S = 0; int last = -1, sel = -1;
    for (int h = 0; h < a.ncomb; ++h) {
      if (!a.good[h]) continue;
      S += m[h]; last = h;
      if (r < S) { sel = h; break; }
    }
    a.sel_hel[i] = sel >= 0 ? sel : last;
  }
  if ((a.sel_col && a.rc) || a.wcol_out) {
    int sel = 0;
    if (a.ncolor > 1) {
      const double* w = a.wpart + (size_t)i * a.nouter * a.ncolor;
      const int ch = a.channel ? a.channel[i >> 5] : 0;
      const unsigned char* allow = ch > 0 ? a.chanflows + (size_t)(ch - 1) * a.ncolor : nullptr;
      double Tc = 0;
      for (int c = 0; c < a.ncolor; ++c) {
        double v = 0; for (int o = 0; o < a.nouter; ++o) v += w[o * a.ncolor + c];
        if (!allow || allow[c]) Tc += v;
        if (a.wcol_out) a.wcol_out[(size_t)i * a.ncolor + c] = v;
      }
      if (a.sel_col && a.rc) {
        double r = a.rc[i] * Tc, S = 0; sel = -1;
        int last = a.ncolor - 1;
        for (int c = 0; c < a.ncolor; ++c) {
          if (allow && !allow[c]) continue;
          double v = 0; for (int o = 0; o < a.nouter; ++o) v += w[o * a.ncolor + c];
          S += v; last = c;
          if (r < S) { sel = c; break; }
        }
        if (sel < 0) sel = last;
      }
    } else if (a.wcol_out) a.wcol_out[i] = T;
    if (a.sel_col && a.rc) a.sel_col[i] = sel;
  }
}

// multichannel: numerator / denominator of an event = its partial sums over the outer-helicity passes and lane chunks, in order
__global__ void mg_chan_finalize_kernel(const double* part, int nevt, int npart, double* num, double* den) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= nevt) return;
  double n = 0, d = 0;
  for (int k = 0; k < npart; ++k) { n += part[((size_t)i * npart + k) * 2]; d += part[((size_t)i * npart + k) * 2 + 1]; }
  if (num) num[i] = n;
  if (den) den[i] = d;
}

// a9: good[h] = 1 iff some event of the batch has |M_h|^2 != 0
// (rel_threshold > 0: |M_h|^2 > rel_threshold * sum_h |M_h|^2 of that event instead -- zeros that arise by cancellation)
__global__ void mg_filter_kernel(const double* mh2, int nevt, int ncomb, double rel_threshold, unsigned int* flags) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= nevt) return;
  double tot = 0;
  if (rel_threshold > 0) for (int h = 0; h < ncomb; ++h) tot += mh2[(size_t)i * ncomb + h];
  for (int h = 0; h < ncomb; ++h) {
    const double v = mh2[(size_t)i * ncomb + h];
    if (rel_threshold > 0 ? (v > rel_threshold * tot) : (v != 0.0)) atomicOr(&flags[h], 1u);
  }
}

// host bridge: a chunk in component-major order raw[row = c-major (4 x npar)][n] -> AOS mom[n][npar][4] ("transposition
// between column- and row-major layout"); MG_LAYOUT_SOA row = c * npar + leg
__global__ void mg_soa_to_aos_kernel(const double* __restrict__ raw, double* __restrict__ mom, int n, int row) {
  const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= (size_t)n * row) return;
  const int r = (int)(i / n), e = (int)(i % n);         // consecutive threads read consecutive events of one row
  const int npar = row / 4, cc = r / npar, leg = r % npar;
  mom[((size_t)e * npar + leg) * 4 + cc] = raw[i];
}
enum { MG_HOST_CHUNKS = 8, MG_HOST_MIN_CHUNK = 8192 };

// FMA-chain microbenchmark: 8 independent chains per thread, register only
template <class T> __global__ void __launch_bounds__(256) mg_fma_kernel(T* out, int iters, T a, T b) {
  T x[8];
#pragma unroll
  for (int k = 0; k < 8; ++k) x[k] = (T)(threadIdx.x + k);
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int u = 0; u < 16; ++u) {
#pragma unroll
      for (int k = 0; k < 8; ++k) x[k] = fma(x[k], a, b);
    }
  }
  T s = 0;
#pragma unroll
  for (int k = 0; k < 8; ++k) s += x[k];
  if (s == (T)123456789) out[0] = s;
}

// =================================================================================================================
// context
// =================================================================================================================
// where one batch's intermediate results live: per-helicity |M_h|^2, colour-flow partial weights, the work-item counter
struct MgWork { double* mh2; double* wpart; unsigned int* counter; };
enum { MG_HOST_LANES = 2 };

struct mg_ctx {
  int process, precision, device;
  mg_sm_params sm;
  double gs_const, gLA, gRA, gLZ, gRZ;      // charged-lepton couplings to the photon and the Z
  double gLAu, gRAu, gLZu, gRZu;            // u-quark couplings (Drell-Yan)
  int npar, ncomb, ncolor, denom, ndiag, namp, nouter, ng;
  int nouter_w;               // outer-helicity partial sums per event in d_wpart (1 when the kernel sums them on chip)
  double mass[8];
  const MgProgramDesc* prog;
  // device copies of the program
  MgTask* d_tasks; uint16_t* d_idx; uint32_t* d_acclist; void* d_colmat; double* d_colfrag; uint16_t* d_flowslot; uint16_t* d_hin; uint16_t* d_hout;
  // multichannel program and its workspace
  const MgProgramDesc* chan; int nchan;
  MgTask* c_tasks; uint16_t* c_idx; uint32_t* c_acclist; uint16_t* c_hin; uint16_t* c_hout; unsigned char* d_chanflows;
  double* d_chanpart; unsigned int* d_chancounter; size_t cap_chan;
  // workspace
  double* d_mh2; double* d_wpart; double* d_scratch; size_t cap_evt;      // d_scratch[nevt]: ME sink of mg_get_last_details
  unsigned char* d_good; unsigned char* d_allgood; unsigned int* d_flags; unsigned int* d_counter;   // d_counter: next work item of the amplitude kernel
  // calls on one context share this workspace: a call on another stream than the previous one first waits for it (ev_done)
  cudaEvent_t ev_done; cudaStream_t last_stream; bool have_last;
  // staging buffers of mg_compute_host
  // mg_compute_host: two lanes, each with its own stream, workspace and staging buffers for one chunk of events
  struct HostLane {
    cudaStream_t st; MgWork w; unsigned int* counter;
    double* mom; double* raw; double* gs; double* rh; double* rc; double* me; int* sh; int* sc;     // raw: chunk as it sits on the host (SOA layout)
  } lane[MG_HOST_LANES];
  size_t lane_cap;            // events per chunk the lanes are sized for
  cudaEvent_t ev_host;        // caller's stream -> lanes
  unsigned char good[128]; int ngood; bool filtered;
  size_t smem_bytes;
  long long launches;
  // optional device timing of the dominant (amplitude) kernel: event pairs recorded on the launching stream
  bool timing; std::vector<cudaEvent_t>* tev;
};
enum { MG_MAX_TIMED_LAUNCHES = 4096 };      // event pairs kept between two mg_kernel_time_ms calls

static thread_local char g_errbuf[320] = "";

#define CUDA_TRY(ctx, expr)                                                                         \
  do {                                                                                              \
    cudaError_t _e = (expr);                                                                        \
    if (_e != cudaSuccess) {                                                                        \
      snprintf(g_errbuf, sizeof(g_errbuf), "CUDA error: %s (%s)", cudaGetErrorString(_e), #expr);   \
      return MG_ECUDA;                                                                              \
    }                                                                                               \
  } while (0)

static void sm_derive(mg_ctx* c) {
  const double PI = 3.14159265358979323846;
  const mg_sm_params& s = c->sm;
  double aEW = 1.0 / s.aEWM1, MZ2 = s.MZ * s.MZ;
  double MW2 = MZ2 / 2 + sqrt(MZ2 * MZ2 / 4 - PI * aEW * MZ2 / (sqrt(2.0) * s.Gf));
  double sw2 = 1 - MW2 / MZ2, ee = sqrt(4 * PI * aEW);
  double sw = sqrt(sw2), cw = sqrt(1 - sw2);
  c->gs_const = sqrt(4 * PI * s.alpha_s);
  c->gLA = -ee; c->gRA = -ee;                      // photon: e Q, Q = -1
  c->gLZ = ee / (sw * cw) * (-0.5 + sw2);          // (e / sw cw)(T3 - Q sw^2)
  c->gRZ = ee / (sw * cw) * sw2;                   // (e / sw cw)(-Q sw^2)
  const double Qu = 2.0 / 3.0;                     // u quark: Q = 2/3, T3 = 1/2
  c->gLAu = ee * Qu; c->gRAu = ee * Qu;
  c->gLZu = ee / (sw * cw) * (0.5 - Qu * sw2); c->gRZu = ee / (sw * cw) * (-Qu * sw2);
}

template <class T> static size_t vm_smem_bytes(const MgProgramDesc* P, bool chan = false) {
  size_t E = P->E, NL = (size_t)P->NC * P->E;
  if (chan) return vm_smem_bytes<T>(P, false) + 2 * NL * sizeof(double);       // channel sums in place of jamp (ncolor = 0 in the descriptor)
  size_t dbl = (8 * 4 * E + ((E + 1) & ~(size_t)1) + P->nthreads) * sizeof(double);
  size_t t = (8 * (size_t)P->nslot * E + ((size_t)1 << P->ng) * MOMSTRIDE * E + (size_t)P->ncolor * 2 * NL + (size_t)(P->ncol + 1) * 2 * NL) * sizeof(T);   // +1: zero column
  return dbl + t;
}

template <class T, class TC, class CFG, bool CHAN = false, class TS = double> static cudaError_t launch_vm_cfg(mg_ctx* c, const VmArgs& a, int grid, cudaStream_t st) {
  size_t smem = CHAN ? vm_smem_bytes<T>(c->chan, true) : vm_smem_bytes<T>(c->prog);
  cudaError_t e = cudaFuncSetAttribute(mg_vm_kernel<T, TC, CFG, CHAN, TS>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (e != cudaSuccess) return e;
  // persistent launch: as many CTAs as fit on the device, each looping over work items
  int occ = 0, dev = 0, nsm = 0;
  e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, mg_vm_kernel<T, TC, CFG, CHAN, TS>, CFG::NT, smem);
  if (e != cudaSuccess) return e;
  cudaGetDevice(&dev);
  cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev);
  int resident = (occ > 0 ? occ : 1) * nsm;
  if (grid > resident) grid = resident;
  mg_vm_kernel<T, TC, CFG, CHAN, TS><<<grid, CFG::NT, smem, st>>>(a);
  return cudaGetLastError();
}
static cudaError_t launch_chan(mg_ctx* c, const VmArgs& a, int grid, cudaStream_t st) {
  switch (c->process) {
    case MG_GG_TT: return launch_vm_cfg<double, double, mgchan2_cfg, true>(c, a, grid, st);
    case MG_GG_TTG: return launch_vm_cfg<double, double, mgchan3_cfg, true>(c, a, grid, st);
    case MG_GG_TTGG: return launch_vm_cfg<double, double, mgchan4_cfg, true>(c, a, grid, st);
    default: return launch_vm_cfg<double, double, mgchan5_cfg, true>(c, a, grid, st);
  }
}
template <class T, class TC> static cudaError_t launch_vm_t(mg_ctx* c, const VmArgs& a, int grid, cudaStream_t st) {
  switch (c->process) {
    case MG_GG_TT: return launch_vm_cfg<T, TC, mgprog2_cfg>(c, a, grid, st);
    case MG_GG_TTG: return launch_vm_cfg<T, TC, mgprog3_cfg>(c, a, grid, st);
    case MG_GG_TTGG: return launch_vm_cfg<T, TC, mgprog4_cfg>(c, a, grid, st);
    case MG_GG_TTGGG: return launch_vm_cfg<T, TC, mgprog5_cfg>(c, a, grid, st);
    case MG_UU_EE: return launch_vm_cfg<T, TC, mgprog6_cfg>(c, a, grid, st);
    case MG_UU_EEG: return launch_vm_cfg<T, TC, mgprog7_cfg>(c, a, grid, st);
    case MG_UU_EEGG: return launch_vm_cfg<T, TC, mgprog8_cfg>(c, a, grid, st);
    default: return launch_vm_cfg<T, TC, mgprog9_cfg>(c, a, grid, st);
  }
}
// FP32 modes: the FP32 programs of gg->ttgg and gg->ttggg (more events per CTA); TS = float is the all-FP32 mode
template <class TS> static cudaError_t launch_vm_f32(mg_ctx* c, const VmArgs& a, int grid, cudaStream_t st) {
  switch (c->process) {
    case MG_GG_TT: return launch_vm_cfg<float, float, mgprog2_cfg, false, TS>(c, a, grid, st);
    case MG_GG_TTG: return launch_vm_cfg<float, float, mgprog3_cfg, false, TS>(c, a, grid, st);
    case MG_GG_TTGG: return launch_vm_cfg<float, float, mgprog4f_cfg, false, TS>(c, a, grid, st);
    case MG_GG_TTGGG: return launch_vm_cfg<float, float, mgprog5f_cfg, false, TS>(c, a, grid, st);
    case MG_UU_EE: return launch_vm_cfg<float, float, mgprog6_cfg, false, TS>(c, a, grid, st);
    case MG_UU_EEG: return launch_vm_cfg<float, float, mgprog7_cfg, false, TS>(c, a, grid, st);
    case MG_UU_EEGG: return launch_vm_cfg<float, float, mgprog8_cfg, false, TS>(c, a, grid, st);
    default: return launch_vm_cfg<float, float, mgprog9_cfg, false, TS>(c, a, grid, st);
  }
}

static int ensure_workspace(mg_ctx* c, int nevt) {
  if ((size_t)nevt <= c->cap_evt) return MG_OK;
  if (c->d_mh2) cudaFree(c->d_mh2);
  if (c->d_wpart) cudaFree(c->d_wpart);
  if (c->d_scratch) cudaFree(c->d_scratch);
  c->d_mh2 = c->d_wpart = c->d_scratch = nullptr; c->cap_evt = 0;
  if (cudaMalloc(&c->d_mh2, (size_t)nevt * c->ncomb * sizeof(double)) != cudaSuccess) { cudaGetLastError(); return MG_ENOMEM; }
  if (cudaMalloc(&c->d_wpart, (size_t)nevt * c->nouter_w * c->ncolor * sizeof(double)) != cudaSuccess) { cudaGetLastError(); return MG_ENOMEM; }
  if (cudaMalloc(&c->d_scratch, (size_t)nevt * sizeof(double)) != cudaSuccess) { cudaGetLastError(); return MG_ENOMEM; }
  c->cap_evt = nevt;
  return MG_OK;
}

// Workspace ordering: every call that touches the context's workspace starts with enter() and ends with leave().
static int enter(mg_ctx* c, cudaStream_t st) {
  if (c->have_last && c->last_stream != st) CUDA_TRY(c, cudaStreamWaitEvent(st, c->ev_done, 0));
  return MG_OK;
}
static int leave(mg_ctx* c, cudaStream_t st) {
  CUDA_TRY(c, cudaEventRecord(c->ev_done, st));
  c->last_stream = st; c->have_last = true;
  return MG_OK;
}

// per-helicity |M_h|^2 and colour-flow partial weights of a batch into the workspace
static int run_amplitudes_impl(mg_ctx* c, const MgWork& w, const double* d_momenta, const double* d_gs, int nevt, int layout, unsigned long long mask, cudaStream_t st);
static int run_amplitudes(mg_ctx* c, const MgWork& w, const double* d_momenta, const double* d_gs, int nevt, int layout, unsigned long long mask, cudaStream_t st,
                          bool timed = true) {
  if (!timed || !c->timing || c->tev->size() >= 2 * MG_MAX_TIMED_LAUNCHES) return run_amplitudes_impl(c, w, d_momenta, d_gs, nevt, layout, mask, st);
  cudaEvent_t e0 = nullptr, e1 = nullptr;
  if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) {
    if (e0) cudaEventDestroy(e0);
    snprintf(g_errbuf, sizeof(g_errbuf), "CUDA error: %s (timing events)", cudaGetErrorString(cudaGetLastError()));
    return MG_ECUDA;
  }
  cudaEventRecord(e0, st);
  int rc = run_amplitudes_impl(c, w, d_momenta, d_gs, nevt, layout, mask, st);
  cudaEventRecord(e1, st);
  if (rc != MG_OK) { cudaEventDestroy(e0); cudaEventDestroy(e1); return rc; }
  c->tev->push_back(e0); c->tev->push_back(e1);
  return rc;
}
static int run_amplitudes_impl(mg_ctx* c, const MgWork& w, const double* d_momenta, const double* d_gs, int nevt, int layout, unsigned long long mask, cudaStream_t st) {
  if (c->process == MG_EE_MUMU) {
    EEArgs a = {d_momenta, nevt, layout, c->sm.MZ, c->sm.WZ, c->gLA, c->gRA, c->gLZ, c->gRZ, w.mh2, mask};
    mg_ee_kernel<<<(nevt + 127) / 128, 128, 0, st>>>(a);
    c->launches++;
    CUDA_TRY(c, cudaGetLastError());
    return MG_OK;
  }
  const MgProgramDesc* P = c->prog;
  VmArgs a;
  a.channel = nullptr; a.good = nullptr; a.chanpart = nullptr;
  a.tasks = c->d_tasks; a.idx = c->d_idx; a.acclist = c->d_acclist; a.colmat = c->d_colmat; a.colfrag = c->d_colfrag; a.flowslot = c->d_flowslot;
  a.hin = c->d_hin; a.hout = c->d_hout; a.momenta = d_momenta; a.gs = d_gs; a.mh2 = w.mh2; a.wpart = w.wpart;
  a.nevt = nevt; a.layout = layout; a.pos_t = P->pos_t; a.pos_tb = P->pos_tb;
  for (int k = 0; k < 33; ++k) a.unitoff[k] = P->unitoff[k];
  a.mt = c->sm.MT; a.wt = c->sm.WT; a.gs_const = c->gs_const; a.inv_colden = 1.0 / P->colden;
  if (P->split && c->precision == MG_FP64) a.inv_colden *= 0.5;       // the J+- form of the colour sum carries a factor 1/2
  if (c->process >= MG_UU_EE) {          // Drell-Yan: massless quark line without width; couplings of the gamma*/Z vertex
    a.mt = 0.0; a.wt = 0.0;
    const double q[10] = {c->gLAu, c->gRAu, c->gLZu, c->gRZu, c->gLA, c->gRA, c->gLZ, c->gRZ, c->sm.MZ, c->sm.WZ};
    for (int k = 0; k < 10; ++k) a.ew[k] = q[k];
  }
  int grid = ((nevt + P->E - 1) / P->E) * P->nouter;
  a.nwork = grid;
  a.counter = w.counter;
  CUDA_TRY(c, cudaMemsetAsync(w.counter, 0, sizeof(unsigned int), st));
  cudaError_t e;
  if (c->precision == MG_FP64) e = launch_vm_t<double, double>(c, a, grid, st);
  else if (c->precision == MG_FP32) e = launch_vm_f32<double>(c, a, grid, st);
  else if (c->precision == MG_FP32_ALL) e = launch_vm_f32<float>(c, a, grid, st);
  else e = launch_vm_t<double, float>(c, a, grid, st);
  c->launches++;
  CUDA_TRY(c, e);
  return MG_OK;
}

static MgWork main_work(const mg_ctx* c) { return MgWork{c->d_mh2, c->d_wpart, c->d_counter}; }

// a1-a10 for one batch into the workspace `w`: amplitude kernel, then helicity sum / selection / store
static int compute_into(mg_ctx* c, const MgWork& w, const double* d_momenta, const double* d_gs, const double* rh, const double* rcol, int nevt,
                        int layout, double* d_me, int* sel_hel, int* sel_col, cudaStream_t st, bool timed) {
  unsigned long long mask = 0;
  for (int h = 0; h < c->ncomb && h < 64; ++h) if (c->good[h]) mask |= 1ull << h;
  int rc = run_amplitudes(c, w, d_momenta, d_gs, nevt, layout, mask, st, timed);
  if (rc) return rc;
  FinArgs f = {w.mh2, w.wpart, c->d_good, rh, rcol, d_me, sel_hel, sel_col, nullptr,
               nevt, c->ncomb, c->ncolor, c->nouter_w, c->denom};
  mg_finalize_kernel<<<(nevt + 127) / 128, 128, 0, st>>>(f);
  c->launches++;
  CUDA_TRY(c, cudaGetLastError());
  return MG_OK;
}

template <class T> static cudaError_t upload(T** dst, const T* src, size_t n) {
  cudaError_t e = cudaMalloc((void**)dst, (n ? n : 1) * sizeof(T));
  if (e != cudaSuccess) return e;
  return n ? cudaMemcpy(*dst, src, n * sizeof(T), cudaMemcpyHostToDevice) : cudaSuccess;
}

// =================================================================================================================
// mg_compute_noalloc: scratch in a file-scope device array (include/mg5b200.h).  Every GPU that loads the library holds
// these MG_NOALLOC_SCRATCH_BYTES until exit.  In host code `mg_noalloc_scratch` is only a host-side stand-in for the
// symbol: its DEVICE address is resolved once per device by cudaGetSymbolAddress (with that device current) and that
// pointer is what the kernels get.  Layout per call: [work-item counter, 256 bytes][mh2: nevt x ncomb][wpart: nevt x nouter_w x ncolor].
// =================================================================================================================
static __device__ __align__(256) unsigned char mg_noalloc_scratch[MG_NOALLOC_SCRATCH_BYTES];
enum { MG_NOALLOC_MAX_DEVICES = 64, MG_NOALLOC_HEADER = 256 };
static unsigned char* g_noalloc_ptr[MG_NOALLOC_MAX_DEVICES];     // device address of mg_noalloc_scratch per device, 0 = not resolved yet

// device address of the scratch array on the context's device (which must be current); no allocation
static int noalloc_scratch_ptr(mg_ctx* c, unsigned char** out) {
  if (c->device < 0 || c->device >= MG_NOALLOC_MAX_DEVICES) { snprintf(g_errbuf, sizeof(g_errbuf), "mg_compute_noalloc: device %d is beyond the %d supported", c->device, (int)MG_NOALLOC_MAX_DEVICES); return MG_EINVAL; }
  if (!g_noalloc_ptr[c->device]) {
    void* p = nullptr;
    CUDA_TRY(c, cudaGetSymbolAddress(&p, mg_noalloc_scratch));
    g_noalloc_ptr[c->device] = static_cast<unsigned char*>(p);
  }
  *out = g_noalloc_ptr[c->device];
  return MG_OK;
}

template <int MODE> static cudaError_t launch_pipes(int grid, size_t smem, double* d, int iters) {
  cudaError_t e = cudaFuncSetAttribute(mg_pipes_kernel<MODE>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (e != cudaSuccess) return e;
  mg_pipes_kernel<MODE><<<grid, 512, smem>>>(d, iters, 1.0000001, 1e-9);
  return cudaGetLastError();
}

extern "C" {

static void free_lanes(mg_ctx* c);

int mg_create(mg_ctx** out, int process, const mg_sm_params* sm, int precision, int device) {
  if (!out || !sm || process < MG_EE_MUMU || process > MG_UU_EEGGG || precision < MG_FP64 || precision > MG_FP32_ALL) {
    snprintf(g_errbuf, sizeof(g_errbuf), "mg_create: invalid argument");
    return MG_EINVAL;
  }
  if (process == MG_EE_MUMU && precision != MG_FP64) { snprintf(g_errbuf, sizeof(g_errbuf), "mg_create: e+e- -> mu+mu- is FP64 only"); return MG_EINVAL; }
  {
    // physical Standard-Model inputs only: masses and widths finite and >= 0 (MZ > 0), couplings > 0, real MW
    const double v[7] = {sm->MZ, sm->WZ, sm->MT, sm->WT, sm->aEWM1, sm->Gf, sm->alpha_s};
    bool ok = true;
    for (int k = 0; k < 7; ++k) ok = ok && std::isfinite(v[k]) && v[k] >= 0;
    ok = ok && sm->MZ > 0 && sm->aEWM1 > 0 && sm->Gf > 0 && sm->alpha_s > 0;
    if (ok) { const double MZ2 = sm->MZ * sm->MZ; ok = MZ2 * MZ2 / 4 - 3.14159265358979323846 / sm->aEWM1 * MZ2 / (sqrt(2.0) * sm->Gf) >= 0; }
    if (!ok) { snprintf(g_errbuf, sizeof(g_errbuf), "mg_create: non-physical Standard-Model parameters"); return MG_EINVAL; }
  }
  int ndev = 0;
  CUDA_TRY(0, cudaGetDeviceCount(&ndev));
  if (device < 0 || device >= ndev) { snprintf(g_errbuf, sizeof(g_errbuf), "mg_create: no CUDA device %d (%d visible)", device, ndev); return MG_EINVAL; }
  CUDA_TRY(0, cudaSetDevice(device));
  mg_ctx* c = new (std::nothrow) mg_ctx();
  if (!c) return MG_ENOMEM;
  memset(c, 0, sizeof(*c));
  c->tev = new std::vector<cudaEvent_t>();
  c->process = process; c->precision = precision; c->device = device; c->sm = *sm;
  sm_derive(c);
  c->ngood = -1;
  if (process == MG_EE_MUMU) {
    c->npar = 4; c->ncomb = 16; c->ncolor = 1; c->denom = 4; c->ndiag = 2; c->namp = 2; c->nouter = 1; c->nouter_w = 1; c->ng = 0;
  } else {
    const bool f32 = precision == MG_FP32 || precision == MG_FP32_ALL;
    const MgProgramDesc* P = f32 ? mg_f32_table[process] : mg_program_table[process];
    c->prog = P; c->ng = P->ng; c->npar = P->npar; c->ncomb = 1 << P->npar; c->ncolor = P->ncolor; c->nouter = P->nouter;
    c->ndiag = P->ndiag; c->namp = P->namp;
    // mg_vm.cuh: with four or more outer passes they run back to back in one CTA and, in the E = 1 form, the flow weights are summed on chip
    c->nouter_w = (P->nouter >= MG_PER_TILE_MIN && P->E == 1 && P->NC == 32 && P->nthreads >= 4 * P->ncolor) ? 1 : P->nouter;
    if (process >= MG_UU_EE) {
      // u u~ -> e+ e- + n g: 2 x 2 spins, 3 x 3 colours, n! for the identical gluons; all external legs massless
      int fact = 1; for (int k = 2; k <= P->ng - 1; ++k) fact *= k;
      c->denom = 36 * fact;
    } else {
      int fact = 1; for (int k = 2; k <= P->ng - 2; ++k) fact *= k;
      c->denom = 256 * fact;
      c->mass[2] = c->mass[3] = sm->MT;
    }
    cudaError_t e = upload(&c->d_tasks, P->tasks, (size_t)P->ntasks);
    if (e == cudaSuccess) e = upload(&c->d_idx, P->idx, (size_t)P->nidx * 8);
    if (e == cudaSuccess) e = upload(&c->d_acclist, P->acclist, (size_t)P->nacclist);
    if (e == cudaSuccess) e = upload(&c->d_hin, P->hin, (size_t)P->NC);
    if (e == cudaSuccess) e = upload(&c->d_hout, P->hout, (size_t)P->nouter);
    // colour-matrix numerators blocked for the colour stage: [row group g][column t][RPT rows], zero padded
    const int NLp = P->NC * P->E, G = P->nthreads / NLp, RPT = (P->ncolor + G - 1) / G;
    size_t nn = (size_t)G * P->ncolor * RPT;
    if (e == cudaSuccess) {
      std::vector<double> m((nn + 3) / 4 * 4, 0.0);       // padded: the kernel stages whole 16-byte words
      for (int g = 0; g < G; ++g) for (int t = 0; t < P->ncolor; ++t) for (int r = 0; r < RPT; ++r) {
        int s = g * RPT + r;
        // symmetric form: C on the diagonal blocks, 2C above them, 0 below (the kernel walks columns t >= g * RPT only)
        double f = t < g * RPT ? 0.0 : (t < (g + 1) * RPT ? 1.0 : 2.0);
        if (s < P->ncolor) m[((size_t)g * P->ncolor + t) * RPT + r] = f * P->colnum[(size_t)s * P->ncolor + t];
      }
      if (precision == MG_FP64) { double* d; e = upload(&d, m.data(), m.size()); c->d_colmat = d; }
      else { std::vector<float> mf(m.begin(), m.end()); float* d; e = upload(&d, mf.data(), mf.size()); c->d_colmat = d; }
    }
    // FP64 tensor-core form (mg_vm.cuh colour stage): numerators of C' = (Caa + Cab) (+) (Caa - Cab) as mma.sync m8n8k4 B fragments.
    // Per non-zero block pair kb_lo(nb) <= kb <= nb of 8 x 8 blocks and k-step ks, lane T holds f * C'[kb*8 + ks*4 + T%4][nb*8 + T/4],
    // f = 1 on the diagonal blocks, 2 above (C' symmetric: the upper block triangle is walked once)
    if (e == cudaSuccess && P->split) {
      const int NB = P->ncolor / 8, half = P->ncolor / 2;
      std::vector<double> fr;
      for (int nb = 0; nb < NB; ++nb) for (int kb = (nb * 8 >= half ? half / 8 : 0); kb <= nb; ++kb) for (int ks = 0; ks < 2; ++ks) for (int T = 0; T < 32; ++T)
        fr.push_back((kb == nb ? 1.0 : 2.0) * P->colprime[(size_t)(kb * 8 + ks * 4 + T % 4) * P->ncolor + nb * 8 + T / 4]);
      e = upload(&c->d_colfrag, fr.data(), fr.size());
    }
    if (e == cudaSuccess) e = upload(&c->d_flowslot, P->flowslot, (size_t)P->ncolor);
    // the multichannel program of the process, its tables and the allowed colour flows per channel
    const MgProgramDesc* Q = mg_chan_table[process];
    c->chan = Q; c->nchan = mg_nchan_table[process];
    if (Q) {
      if (e == cudaSuccess) e = upload(&c->c_tasks, Q->tasks, (size_t)Q->ntasks);
      if (e == cudaSuccess) e = upload(&c->c_idx, Q->idx, (size_t)Q->nidx * 8);
      if (e == cudaSuccess) e = upload(&c->c_acclist, Q->acclist, (size_t)Q->nacclist);
      if (e == cudaSuccess) e = upload(&c->c_hin, Q->hin, (size_t)Q->NC);
      if (e == cudaSuccess) e = upload(&c->c_hout, Q->hout, (size_t)Q->nouter);
      if (e == cudaSuccess) e = upload(&c->d_chanflows, mg_chanflows_table[process], (size_t)c->nchan * P->ncolor);
      if (e == cudaSuccess && cudaMalloc(&c->d_chancounter, sizeof(unsigned int)) != cudaSuccess) e = cudaErrorMemoryAllocation;
    }
    if (e != cudaSuccess) { snprintf(g_errbuf, sizeof(g_errbuf), "CUDA error: %s (program upload)", cudaGetErrorString(e)); mg_destroy(c); return MG_ECUDA; }
    c->smem_bytes = f32 ? vm_smem_bytes<float>(P) : vm_smem_bytes<double>(P);
  }
  if (cudaMalloc(&c->d_good, 128) != cudaSuccess || cudaMalloc(&c->d_allgood, 128) != cudaSuccess || cudaMalloc(&c->d_flags, 128 * sizeof(unsigned int)) != cudaSuccess ||
      cudaMalloc(&c->d_counter, sizeof(unsigned int)) != cudaSuccess || cudaMemset(c->d_allgood, 1, 128) != cudaSuccess ||
      cudaEventCreateWithFlags(&c->ev_done, cudaEventDisableTiming) != cudaSuccess) { cudaGetLastError(); mg_destroy(c); return MG_ENOMEM; }
  *out = c;
  return MG_OK;
}

int mg_destroy(mg_ctx* c) {
  if (!c) return MG_OK;
  cudaSetDevice(c->device);
  cudaFree(c->d_tasks); cudaFree(c->d_idx); cudaFree(c->d_acclist); cudaFree(c->d_colmat); cudaFree(c->d_colfrag); cudaFree(c->d_flowslot);
  cudaFree(c->d_hin); cudaFree(c->d_hout); cudaFree(c->d_mh2); cudaFree(c->d_wpart); cudaFree(c->d_scratch); cudaFree(c->d_good); cudaFree(c->d_allgood);
  cudaFree(c->d_flags); cudaFree(c->d_counter);
  if (c->ev_done) cudaEventDestroy(c->ev_done);
  cudaFree(c->c_tasks); cudaFree(c->c_idx); cudaFree(c->c_acclist); cudaFree(c->c_hin); cudaFree(c->c_hout); cudaFree(c->d_chanflows);
  cudaFree(c->d_chanpart); cudaFree(c->d_chancounter);
  free_lanes(c);
  for (int k = 0; k < MG_HOST_LANES; ++k) if (c->lane[k].st) cudaStreamDestroy(c->lane[k].st);
  if (c->ev_host) cudaEventDestroy(c->ev_host);
  if (c->tev) { for (cudaEvent_t e : *c->tev) cudaEventDestroy(e); delete c->tev; }
  delete c;
  return MG_OK;
}

int mg_get_info(const mg_ctx* c, mg_info* o) {
  if (!c || !o) return MG_EINVAL;
  memset(o, 0, sizeof(*o));
  o->npar = c->npar; o->ndiag = c->ndiag; o->namp = c->namp; o->ncolor = c->ncolor; o->ncomb = c->ncomb; o->ngood = c->ngood; o->denom = c->denom;
  for (int k = 0; k < 8; ++k) o->mass[k] = c->mass[k];
  o->nchannel = c->nchan;
  if (c->prog) { o->flops_per_event = c->prog->flops_exec; o->flops_per_event_canonical = c->prog->flops_canonical; }
  else { o->flops_per_event = mg_ee_flops_exec; o->flops_per_event_canonical = mg_ee_flops_canonical; }   // counted by the emitter
  return MG_OK;
}

int mg_sample_rambo(mg_ctx* c, unsigned long long seed, unsigned long long first, int nevt, double sqrt_s, int layout,
                    double* d_momenta, double* d_weight, void* stream) {
  if (!c || !d_momenta || nevt < 0 || sqrt_s <= 0 || (layout != MG_LAYOUT_AOS && layout != MG_LAYOUT_AOSOA) ||
      (layout == MG_LAYOUT_AOSOA && nevt % MG_AOSOA_V)) { snprintf(g_errbuf, sizeof(g_errbuf), "mg_sample_rambo: invalid argument"); return MG_EINVAL; }
  {
    double summ = 0;
    for (int k = 2; k < c->npar; ++k) summ += c->mass[k];
    if (!std::isfinite(sqrt_s) || sqrt_s <= summ) { snprintf(g_errbuf, sizeof(g_errbuf), "mg_sample_rambo: sqrt_s = %g is not above the sum of the final-state masses %g", sqrt_s, summ); return MG_EINVAL; }
  }
  if (nevt == 0) return MG_OK;
  CUDA_TRY(c, cudaSetDevice(c->device));
  RamboArgs a; a.seed = seed; a.first = first; a.nevt = nevt; a.nf = c->npar - 2; a.layout = layout; a.E = sqrt_s; a.p = d_momenta; a.w = d_weight;
  for (int k = 0; k < 6; ++k) a.mass[k] = k + 2 < 8 ? c->mass[k + 2] : 0.0;
  mg_rambo_kernel<<<(nevt + 127) / 128, 128, 0, (cudaStream_t)stream>>>(a);
  c->launches++;
  CUDA_TRY(c, cudaGetLastError());
  return MG_OK;
}

int mg_sample_uniforms(mg_ctx* c, unsigned long long seed, unsigned long long first, int nevt, double* rh, double* rc, void* stream) {
  if (!c || nevt < 0) { snprintf(g_errbuf, sizeof(g_errbuf), "mg_sample_uniforms: invalid argument"); return MG_EINVAL; }
  if (nevt == 0 || (!rh && !rc)) return MG_OK;
  CUDA_TRY(c, cudaSetDevice(c->device));
  mg_uniforms_kernel<<<(nevt + 255) / 256, 256, 0, (cudaStream_t)stream>>>(seed, first, nevt, rh, rc);
  c->launches++;
  CUDA_TRY(c, cudaGetLastError());
  return MG_OK;
}

static int check_batch(mg_ctx* c, const double* d_momenta, int nevt, int layout, const char* who) {
  if (!c || !d_momenta || nevt < 0 || (layout != MG_LAYOUT_AOS && layout != MG_LAYOUT_AOSOA) || (layout == MG_LAYOUT_AOSOA && nevt % MG_AOSOA_V)) {
    snprintf(g_errbuf, sizeof(g_errbuf), "%s: invalid argument", who);
    return MG_EINVAL;
  }
  return MG_OK;
}

static int install_mask(mg_ctx* c, const unsigned char* mask, cudaStream_t st) {
  c->ngood = 0;
  for (int h = 0; h < c->ncomb; ++h) { c->good[h] = mask[h] ? 1 : 0; c->ngood += c->good[h]; }
  CUDA_TRY(c, cudaMemcpyAsync(c->d_good, c->good, c->ncomb, cudaMemcpyHostToDevice, st));
  CUDA_TRY(c, cudaStreamSynchronize(st));
  c->filtered = true;
  return MG_OK;
}

int mg_filter_helicities(mg_ctx* c, const double* d_momenta, const double* d_gs, int nevt, int layout, double rel_threshold,
                         int* ngood_out, unsigned char* h_good_out, void* stream) {
  int rc = check_batch(c, d_momenta, nevt, layout, "mg_filter_helicities");
  if (rc) return rc;
  if (nevt == 0) { snprintf(g_errbuf, sizeof(g_errbuf), "mg_filter_helicities: empty batch"); return MG_EINVAL; }
  if (!(rel_threshold >= 0) || rel_threshold >= 1) { snprintf(g_errbuf, sizeof(g_errbuf), "mg_filter_helicities: rel_threshold must be in [0, 1)"); return MG_EINVAL; }
  cudaStream_t st = (cudaStream_t)stream;
  CUDA_TRY(c, cudaSetDevice(c->device));
  rc = ensure_workspace(c, nevt);
  if (rc) return rc;
  if ((rc = enter(c, st)) != MG_OK) return rc;
  rc = run_amplitudes(c, main_work(c), d_momenta, d_gs, nevt, layout, ~0ull, st);
  if (rc) return rc;
  CUDA_TRY(c, cudaMemsetAsync(c->d_flags, 0, 128 * sizeof(unsigned int), st));
  mg_filter_kernel<<<(nevt + 127) / 128, 128, 0, st>>>(c->d_mh2, nevt, c->ncomb, rel_threshold, c->d_flags);
  c->launches++;
  CUDA_TRY(c, cudaGetLastError());
  unsigned int flags[128];
  CUDA_TRY(c, cudaMemcpyAsync(flags, c->d_flags, c->ncomb * sizeof(unsigned int), cudaMemcpyDeviceToHost, st));
  CUDA_TRY(c, cudaStreamSynchronize(st));
  unsigned char mask[128];
  for (int h = 0; h < c->ncomb; ++h) mask[h] = flags[h] ? 1 : 0;
  if ((rc = install_mask(c, mask, st)) != MG_OK) return rc;
  if ((rc = leave(c, st)) != MG_OK) return rc;
  if (ngood_out) *ngood_out = c->ngood;
  if (h_good_out) memcpy(h_good_out, c->good, c->ncomb);
  return MG_OK;
}

int mg_set_good_helicities(mg_ctx* c, const unsigned char* h_mask, void* stream) {
  if (!c || !h_mask) { snprintf(g_errbuf, sizeof(g_errbuf), "mg_set_good_helicities: invalid argument"); return MG_EINVAL; }
  int n = 0;
  for (int h = 0; h < c->ncomb; ++h) { if (h_mask[h] > 1) { snprintf(g_errbuf, sizeof(g_errbuf), "mg_set_good_helicities: mask bytes must be 0 or 1"); return MG_EINVAL; } n += h_mask[h]; }
  if (n == 0) { snprintf(g_errbuf, sizeof(g_errbuf), "mg_set_good_helicities: empty mask"); return MG_EINVAL; }
  cudaStream_t st = (cudaStream_t)stream;
  CUDA_TRY(c, cudaSetDevice(c->device));
  int rc = enter(c, st);
  if (rc) return rc;
  if ((rc = install_mask(c, h_mask, st)) != MG_OK) return rc;
  return leave(c, st);
}

int mg_compute(mg_ctx* c, const double* d_momenta, const double* d_gs, const double* rh, const double* rcol, int nevt, int layout,
               double* d_me, int* sel_hel, int* sel_col, void* stream) {
  int rc = check_batch(c, d_momenta, nevt, layout, "mg_compute");
  if (rc) return rc;
  if (!d_me) { snprintf(g_errbuf, sizeof(g_errbuf), "mg_compute: d_me is NULL"); return MG_EINVAL; }
  if (!c->filtered) { snprintf(g_errbuf, sizeof(g_errbuf), "mg_compute: call mg_filter_helicities first"); return MG_ENOTFILTERED; }
  if (nevt == 0) return MG_OK;
  cudaStream_t st = (cudaStream_t)stream;
  CUDA_TRY(c, cudaSetDevice(c->device));
  rc = ensure_workspace(c, nevt);
  if (rc) return rc;
  if ((rc = enter(c, st)) != MG_OK) return rc;
  if ((rc = compute_into(c, main_work(c), d_momenta, d_gs, rh, rcol, nevt, layout, d_me, sel_hel, sel_col, st, true)) != MG_OK) return rc;
  return leave(c, st);
}

int mg_compute_noalloc(mg_ctx* c, const double* d_momenta, const double* d_gs, const double* rh, const double* rcol, int nevt, int layout,
                       double* d_me, int* sel_hel, int* sel_col, void* stream) {
  int rc = check_batch(c, d_momenta, nevt, layout, "mg_compute_noalloc");
  if (rc) return rc;
  if (!d_me) { snprintf(g_errbuf, sizeof(g_errbuf), "mg_compute_noalloc: d_me is NULL"); return MG_EINVAL; }
  if (!c->filtered) { snprintf(g_errbuf, sizeof(g_errbuf), "mg_compute_noalloc: call mg_filter_helicities or mg_set_good_helicities first"); return MG_ENOTFILTERED; }
  const size_t per_evt = ((size_t)c->ncomb + (size_t)c->nouter_w * c->ncolor) * sizeof(double);
  const size_t max_evt = ((size_t)MG_NOALLOC_SCRATCH_BYTES - MG_NOALLOC_HEADER) / per_evt;
  if ((size_t)nevt > max_evt) {
    snprintf(g_errbuf, sizeof(g_errbuf), "mg_compute_noalloc: nevt = %d needs %zu bytes of scratch but the static array holds %zu: at most %zu events "
             "per call for this process (use mg_compute, or split the batch)", nevt, MG_NOALLOC_HEADER + (size_t)nevt * per_evt, (size_t)MG_NOALLOC_SCRATCH_BYTES, max_evt);
    return MG_EINVAL;
  }
  if (nevt == 0) return MG_OK;
  cudaStream_t st = (cudaStream_t)stream;
  CUDA_TRY(c, cudaSetDevice(c->device));
  unsigned char* base = nullptr;
  if ((rc = noalloc_scratch_ptr(c, &base)) != MG_OK) return rc;
  if ((rc = enter(c, st)) != MG_OK) return rc;
  // the kernels of mg_compute, pointed at the static scratch instead of the context's workspace: the counter is zeroed on the
  // stream by the amplitude launch, mh2 and wpart are fully rewritten (no kernel-timing events: creating them allocates)
  MgWork w;
  w.counter = reinterpret_cast<unsigned int*>(base);
  w.mh2 = reinterpret_cast<double*>(base + MG_NOALLOC_HEADER);
  w.wpart = w.mh2 + (size_t)nevt * c->ncomb;
  if ((rc = compute_into(c, w, d_momenta, d_gs, rh, rcol, nevt, layout, d_me, sel_hel, sel_col, st, false)) != MG_OK) return rc;
  return leave(c, st);
}

int mg_compute_multichannel(mg_ctx* c, const double* d_momenta, const double* d_gs, const double* rh, const double* rcol, const int* d_channel,
                            int nevt, int layout, double* d_me, int* sel_hel, int* sel_col, double* d_num, double* d_den, void* stream) {
  int rc = check_batch(c, d_momenta, nevt, layout, "mg_compute_multichannel");
  if (rc) return rc;
  if (!c->chan) { snprintf(g_errbuf, sizeof(g_errbuf), "mg_compute_multichannel: the process has no multichannel program (g g -> t t~ + gluons only)"); return MG_EINVAL; }
  if (!d_me || !d_channel || !d_num || !d_den) { snprintf(g_errbuf, sizeof(g_errbuf), "mg_compute_multichannel: d_me, d_channel, d_num and d_den must not be NULL"); return MG_EINVAL; }
  if (!c->filtered) { snprintf(g_errbuf, sizeof(g_errbuf), "mg_compute_multichannel: call mg_filter_helicities first"); return MG_ENOTFILTERED; }
  if (nevt == 0) return MG_OK;
  cudaStream_t st = (cudaStream_t)stream;
  CUDA_TRY(c, cudaSetDevice(c->device));
  rc = ensure_workspace(c, nevt);
  if (rc) return rc;
  const MgProgramDesc* Q = c->chan;
  const int npart = Q->nouter * (Q->NC * Q->E / 32);
  if ((size_t)nevt > c->cap_chan) {
    cudaFree(c->d_chanpart); c->d_chanpart = nullptr; c->cap_chan = 0;
    if (cudaMalloc(&c->d_chanpart, (size_t)nevt * npart * 2 * sizeof(double)) != cudaSuccess) { cudaGetLastError(); return MG_ENOMEM; }
    c->cap_chan = nevt;
  }
  if ((rc = enter(c, st)) != MG_OK) return rc;
  // (1) the matrix element as in mg_compute, the colour selected among the flows of the event's channel
  const MgWork w = main_work(c);
  unsigned long long mask = 0;
  for (int h = 0; h < c->ncomb && h < 64; ++h) if (c->good[h]) mask |= 1ull << h;
  if ((rc = run_amplitudes(c, w, d_momenta, d_gs, nevt, layout, mask, st)) != MG_OK) return rc;
  FinArgs f = {w.mh2, w.wpart, c->d_good, rh, rcol, d_me, sel_hel, sel_col, nullptr,
               nevt, c->ncomb, c->ncolor, c->nouter_w, c->denom, d_channel, c->d_chanflows};
  mg_finalize_kernel<<<(nevt + 127) / 128, 128, 0, st>>>(f);
  c->launches++;
  CUDA_TRY(c, cudaGetLastError());
  // (2) the channel sums: the multichannel program (one amplitude column per diagram without four-gluon vertices), always FP64
  VmArgs a;
  a.tasks = c->c_tasks; a.idx = c->c_idx; a.acclist = c->c_acclist; a.colmat = nullptr; a.colfrag = nullptr; a.flowslot = nullptr;
  a.hin = c->c_hin; a.hout = c->c_hout; a.momenta = d_momenta; a.gs = d_gs; a.mh2 = nullptr; a.wpart = nullptr;
  a.nevt = nevt; a.layout = layout; a.pos_t = Q->pos_t; a.pos_tb = Q->pos_tb;
  for (int k = 0; k < 33; ++k) a.unitoff[k] = Q->unitoff[k];
  a.mt = c->sm.MT; a.wt = c->sm.WT; a.gs_const = c->gs_const; a.inv_colden = 0;
  a.nwork = ((nevt + Q->E - 1) / Q->E) * Q->nouter;
  a.counter = c->d_chancounter; a.channel = d_channel; a.good = c->d_good; a.chanpart = c->d_chanpart;
  CUDA_TRY(c, cudaMemsetAsync(c->d_chancounter, 0, sizeof(unsigned int), st));
  cudaError_t e = launch_chan(c, a, a.nwork, st);
  c->launches++;
  CUDA_TRY(c, e);
  mg_chan_finalize_kernel<<<(nevt + 127) / 128, 128, 0, st>>>(c->d_chanpart, nevt, npart, d_num, d_den);
  c->launches++;
  CUDA_TRY(c, cudaGetLastError());
  return leave(c, st);
}

static void free_lanes(mg_ctx* c) {
  for (int k = 0; k < MG_HOST_LANES; ++k) {
    mg_ctx::HostLane& L = c->lane[k];
    cudaFree(L.w.mh2); cudaFree(L.w.wpart); cudaFree(L.w.counter);
    cudaFree(L.mom); cudaFree(L.raw); cudaFree(L.gs); cudaFree(L.rh); cudaFree(L.rc); cudaFree(L.me); cudaFree(L.sh); cudaFree(L.sc);
    cudaStream_t st = L.st;
    memset(&L, 0, sizeof(L));
    L.st = st;
  }
  c->lane_cap = 0;
}

// lanes sized for chunks of `chunk` events; streams and the hand-over event are created on first use and kept
static int ensure_lanes(mg_ctx* c, size_t chunk) {
  for (int k = 0; k < MG_HOST_LANES; ++k)
    if (!c->lane[k].st) CUDA_TRY(c, cudaStreamCreateWithFlags(&c->lane[k].st, cudaStreamNonBlocking));
  if (!c->ev_host) CUDA_TRY(c, cudaEventCreateWithFlags(&c->ev_host, cudaEventDisableTiming));
  if (chunk <= c->lane_cap) return MG_OK;
  free_lanes(c);
  const size_t nm = chunk * c->npar * 4 * sizeof(double);
  for (int k = 0; k < MG_HOST_LANES; ++k) {
    mg_ctx::HostLane& L = c->lane[k];
    if (cudaMalloc(&L.w.mh2, chunk * c->ncomb * sizeof(double)) != cudaSuccess || cudaMalloc(&L.w.wpart, chunk * c->nouter_w * c->ncolor * sizeof(double)) != cudaSuccess ||
        cudaMalloc(&L.w.counter, sizeof(unsigned int)) != cudaSuccess || cudaMalloc(&L.mom, nm) != cudaSuccess || cudaMalloc(&L.raw, nm) != cudaSuccess ||
        cudaMalloc(&L.gs, chunk * sizeof(double)) != cudaSuccess || cudaMalloc(&L.rh, chunk * sizeof(double)) != cudaSuccess ||
        cudaMalloc(&L.rc, chunk * sizeof(double)) != cudaSuccess || cudaMalloc(&L.me, chunk * sizeof(double)) != cudaSuccess ||
        cudaMalloc(&L.sh, chunk * sizeof(int)) != cudaSuccess || cudaMalloc(&L.sc, chunk * sizeof(int)) != cudaSuccess) {
      cudaGetLastError(); free_lanes(c); return MG_ENOMEM;
    }
  }
  c->lane_cap = chunk;
  return MG_OK;
}

int mg_compute_host(mg_ctx* c, const double* h_momenta, const double* h_gs, const double* h_rh, const double* h_rc, int nevt, int layout,
                    double* h_me, int* h_sel_hel, int* h_sel_col, void* stream) {
  if (!c || !h_momenta || nevt < 0 || (layout != MG_LAYOUT_AOS && layout != MG_LAYOUT_AOSOA && layout != MG_LAYOUT_SOA) ||
      (layout == MG_LAYOUT_AOSOA && nevt % MG_AOSOA_V)) { snprintf(g_errbuf, sizeof(g_errbuf), "mg_compute_host: invalid argument"); return MG_EINVAL; }
  if (!h_me) { snprintf(g_errbuf, sizeof(g_errbuf), "mg_compute_host: h_me is NULL"); return MG_EINVAL; }
  if (!c->filtered) { snprintf(g_errbuf, sizeof(g_errbuf), "mg_compute_host: call mg_filter_helicities first"); return MG_ENOTFILTERED; }
  if (nevt == 0) return MG_OK;
  cudaStream_t st = (cudaStream_t)stream;
  CUDA_TRY(c, cudaSetDevice(c->device));
  // chunks of whole AOSOA pages: about MG_HOST_CHUNKS per batch, never below MG_HOST_MIN_CHUNK events (a small batch is one chunk)
  size_t chunk = ((size_t)nevt + MG_HOST_CHUNKS - 1) / MG_HOST_CHUNKS;
  if (chunk < MG_HOST_MIN_CHUNK) chunk = MG_HOST_MIN_CHUNK;
  chunk = (chunk + MG_AOSOA_V - 1) / MG_AOSOA_V * MG_AOSOA_V;
  int rc = ensure_lanes(c, chunk);
  if (rc) return rc;
  if ((rc = enter(c, st)) != MG_OK) return rc;
  CUDA_TRY(c, cudaEventRecord(c->ev_host, st));             // the lanes start after what the caller queued on its stream
  for (int k = 0; k < MG_HOST_LANES; ++k) CUDA_TRY(c, cudaStreamWaitEvent(c->lane[k].st, c->ev_host, 0));
  const size_t row = (size_t)c->npar * 4;
  const bool want_sh = h_rh && h_sel_hel, want_sc = h_rc && h_sel_col;
  int k = 0;
  for (size_t off = 0; off < (size_t)nevt; off += chunk, ++k) {
    const size_t n = (size_t)nevt - off < chunk ? (size_t)nevt - off : chunk;
    mg_ctx::HostLane& L = c->lane[k % MG_HOST_LANES];
    // one copy per buffer per chunk; the lane's stream orders chunk k + 2 behind chunk k, the other lane's copies overlap this
    // lane's kernels (the host side is what limits event generation once the matrix element is fast)
    int dev_layout = layout;
    if (layout == MG_LAYOUT_SOA) {
      CUDA_TRY(c, cudaMemcpy2DAsync(L.raw, n * sizeof(double), h_momenta + off, (size_t)nevt * sizeof(double), n * sizeof(double), row, cudaMemcpyHostToDevice, L.st));
      mg_soa_to_aos_kernel<<<(unsigned)((n * row + 255) / 256), 256, 0, L.st>>>(L.raw, L.mom, (int)n, (int)row);
      c->launches++;
      CUDA_TRY(c, cudaGetLastError());
      dev_layout = MG_LAYOUT_AOS;
    } else {
      CUDA_TRY(c, cudaMemcpyAsync(L.mom, h_momenta + off * row, n * row * sizeof(double), cudaMemcpyHostToDevice, L.st));   // AOS and AOSOA: contiguous
    }
    if (h_gs) CUDA_TRY(c, cudaMemcpyAsync(L.gs, h_gs + off, n * sizeof(double), cudaMemcpyHostToDevice, L.st));
    if (h_rh) CUDA_TRY(c, cudaMemcpyAsync(L.rh, h_rh + off, n * sizeof(double), cudaMemcpyHostToDevice, L.st));
    if (h_rc) CUDA_TRY(c, cudaMemcpyAsync(L.rc, h_rc + off, n * sizeof(double), cudaMemcpyHostToDevice, L.st));
    rc = compute_into(c, L.w, L.mom, h_gs ? L.gs : nullptr, h_rh ? L.rh : nullptr, h_rc ? L.rc : nullptr, (int)n, dev_layout, L.me,
                      want_sh ? L.sh : nullptr, want_sc ? L.sc : nullptr, L.st, false);
    if (rc) return rc;
    CUDA_TRY(c, cudaMemcpyAsync(h_me + off, L.me, n * sizeof(double), cudaMemcpyDeviceToHost, L.st));
    if (want_sh) CUDA_TRY(c, cudaMemcpyAsync(h_sel_hel + off, L.sh, n * sizeof(int), cudaMemcpyDeviceToHost, L.st));
    if (want_sc) CUDA_TRY(c, cudaMemcpyAsync(h_sel_col + off, L.sc, n * sizeof(int), cudaMemcpyDeviceToHost, L.st));
  }
  for (int q = 0; q < MG_HOST_LANES; ++q) CUDA_TRY(c, cudaStreamSynchronize(c->lane[q].st));
  return leave(c, st);
}

int mg_get_last_details(mg_ctx* c, int nevt, double* d_mh2, double* d_wcol, void* stream) {
  if (!c || nevt < 0 || (size_t)nevt > c->cap_evt) { snprintf(g_errbuf, sizeof(g_errbuf), "mg_get_last_details: invalid argument"); return MG_EINVAL; }
  if (nevt == 0) return MG_OK;
  cudaStream_t st = (cudaStream_t)stream;
  CUDA_TRY(c, cudaSetDevice(c->device));
  int rc = enter(c, st);
  if (rc) return rc;
  if (d_mh2) CUDA_TRY(c, cudaMemcpyAsync(d_mh2, c->d_mh2, (size_t)nevt * c->ncomb * sizeof(double), cudaMemcpyDeviceToDevice, st));
  if (d_wcol) {
    // the flow weights from the partial sums: a selection-free finalize pass (all-ones mask, ME into the context's scratch)
    FinArgs f = {c->d_mh2, c->d_wpart, c->d_allgood, nullptr, nullptr, c->d_scratch, nullptr, nullptr, d_wcol,
                 nevt, c->ncomb, c->ncolor, c->nouter_w, c->denom};
    mg_finalize_kernel<<<(nevt + 127) / 128, 128, 0, st>>>(f);
    c->launches++;
    CUDA_TRY(c, cudaGetLastError());
  }
  return leave(c, st);
}

int mg_measure_fma_peak(mg_ctx* c, int precision, double millis, double* out) {
  if (!c || !out || (precision != MG_FP64 && precision != MG_FP32)) { snprintf(g_errbuf, sizeof(g_errbuf), "mg_measure_fma_peak: invalid argument"); return MG_EINVAL; }
  CUDA_TRY(c, cudaSetDevice(c->device));
  cudaDeviceProp prop;
  CUDA_TRY(c, cudaGetDeviceProperties(&prop, c->device));
  int grid = prop.multiProcessorCount * 8, block = 256;
  void* d = nullptr;
  CUDA_TRY(c, cudaMalloc(&d, 64));
  cudaEvent_t e0, e1;
  CUDA_TRY(c, cudaEventCreate(&e0)); CUDA_TRY(c, cudaEventCreate(&e1));
  int iters = 2000;
  double best = 0;
  for (int rep = 0; rep < 6; ++rep) {
    CUDA_TRY(c, cudaEventRecord(e0));
    if (precision == MG_FP64) mg_fma_kernel<double><<<grid, block>>>((double*)d, iters, 1.0000001, 1e-9);
    else mg_fma_kernel<float><<<grid, block>>>((float*)d, iters, 1.0000001f, 1e-9f);
    c->launches++;
    CUDA_TRY(c, cudaEventRecord(e1));
    CUDA_TRY(c, cudaEventSynchronize(e1));
    float ms = 0; CUDA_TRY(c, cudaEventElapsedTime(&ms, e0, e1));
    double flops = 2.0 * 8 * 16 * (double)iters * grid * block;
    double tf = flops / (ms * 1e-3) / 1e12;
    if (rep >= 1 && tf > best) best = tf;
    if (rep == 0 && ms > 0) { double scale = millis / ms; if (scale < 0.05) scale = 0.05; if (scale > 50) scale = 50; iters = (int)(iters * scale) + 1; }
  }
  cudaEventDestroy(e0); cudaEventDestroy(e1); cudaFree(d);
  *out = best;
  return MG_OK;
}

int mg_measure_fp64_pipes(mg_ctx* c, int mode, double millis, double* out) {
  if (!c || !out || mode < 0 || mode > 5) { snprintf(g_errbuf, sizeof(g_errbuf), "mg_measure_fp64_pipes: invalid argument"); return MG_EINVAL; }
  CUDA_TRY(c, cudaSetDevice(c->device));
  cudaDeviceProp prop;
  CUDA_TRY(c, cudaGetDeviceProperties(&prop, c->device));
  const int grid = prop.multiProcessorCount;
  const size_t smem = mode == 4 ? (size_t)(MG_PIPES_K * 64 + 225 * 64) * 8 : mode == 5 ? (size_t)(MG_PIPES_K * 64 + MG_PIPES_K * MG_PIPES_K) * 8 : 0;
  void* d = nullptr;
  CUDA_TRY(c, cudaMalloc(&d, 64));
  cudaEvent_t e0, e1;
  CUDA_TRY(c, cudaEventCreate(&e0)); CUDA_TRY(c, cudaEventCreate(&e1));
  int iters = mode <= 3 ? 2000 : 20;
  double best_ms = 0; int best_iters = 1;
  cudaError_t le = cudaSuccess;
  for (int rep = 0; rep < 6 && le == cudaSuccess; ++rep) {
    cudaEventRecord(e0);
    switch (mode) {
      case 0: le = launch_pipes<0>(grid, smem, (double*)d, iters); break;
      case 1: le = launch_pipes<1>(grid, smem, (double*)d, iters); break;
      case 2: le = launch_pipes<2>(grid, smem, (double*)d, iters); break;
      case 3: le = launch_pipes<3>(grid, smem, (double*)d, iters); break;
      case 4: le = launch_pipes<4>(grid, smem, (double*)d, iters); break;
      default: le = launch_pipes<5>(grid, smem, (double*)d, iters); break;
    }
    c->launches++;
    cudaEventRecord(e1);
    if (le == cudaSuccess) le = cudaEventSynchronize(e1);
    float ms = 0;
    if (le == cudaSuccess) le = cudaEventElapsedTime(&ms, e0, e1);
    if (rep >= 1 && (best_ms == 0 || ms / iters < best_ms / best_iters)) { best_ms = ms; best_iters = iters; }
    if (rep == 0 && ms > 0) { double scale = millis / ms; if (scale < 0.05) scale = 0.05; if (scale > 200) scale = 200; iters = (int)(iters * scale) + 1; }
  }
  cudaEventDestroy(e0); cudaEventDestroy(e1); cudaFree(d);
  if (le != cudaSuccess) { snprintf(g_errbuf, sizeof(g_errbuf), "CUDA error: %s (mg_measure_fp64_pipes)", cudaGetErrorString(le)); return MG_ECUDA; }
  double ff, mf;
  mg_pipes_flops(mode, &ff, &mf);
  const double sec = best_ms * 1e-3 / best_iters;
  out[0] = ff * grid / sec / 1e12; out[1] = mf * grid / sec / 1e12; out[2] = best_ms / best_iters;
  return MG_OK;
}


long long mg_launch_count(const mg_ctx* c) { return c ? c->launches : 0; }

int mg_enable_kernel_timing(mg_ctx* c, int on) {
  if (!c) return MG_EINVAL;
  c->timing = on != 0;
  return MG_OK;
}

int mg_kernel_time_ms(mg_ctx* c, double* total_ms, long long* nlaunch) {
  if (!c || !total_ms || !nlaunch) return MG_EINVAL;
  CUDA_TRY(c, cudaSetDevice(c->device));
  double tot = 0; long long n = 0;
  for (size_t k = 0; k + 1 < c->tev->size(); k += 2) {
    float ms = 0;
    CUDA_TRY(c, cudaEventSynchronize((*c->tev)[k + 1]));
    CUDA_TRY(c, cudaEventElapsedTime(&ms, (*c->tev)[k], (*c->tev)[k + 1]));
    tot += ms; ++n;
    cudaEventDestroy((*c->tev)[k]); cudaEventDestroy((*c->tev)[k + 1]);
  }
  c->tev->clear();
  *total_ms = tot; *nlaunch = n;
  return MG_OK;
}

const char* mg_strerror(int code) {
  switch (code) {
    case MG_OK: return "success";
    case MG_EINVAL: return g_errbuf[0] ? g_errbuf : "invalid argument";
    case MG_ENOTFILTERED: return "mg_compute called before mg_filter_helicities";
    case MG_ECUDA: return g_errbuf[0] ? g_errbuf : "CUDA error";
    case MG_ENOMEM: return "out of device memory";
    default: return "unknown error code";
  }
}

}  // extern "C"
