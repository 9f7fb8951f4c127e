// ORACLE — TEST INFRASTRUCTURE ONLY.
//
// Plain, slow, fp64, one-chain-at-a-time CPU restatement of the hot path of
// "Posterior sampling in the Age of Emulators" (arxiv/paper_2606_04895, PAPER.md), written from
// the paper's equations and the readings listed in DESIGN.md / SURVEY.md §8(c).  It shares no
// code, header, table or helper with the CUDA library under paper_2606_04895_b200/csrc/.  Only
// tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may load
// it.  It is never tuned for speed: scalar loops, no BLAS, no blocking, no fast-math; OpenMP
// `parallel for` over independent chains only.
//
// Parity pins (tests/test_oracle_*.py):  Philox known-answer vectors; transforms' closed forms;
// MLP vs torch fp64 Linear stack and autograd; finite differences; Gaussian closed-form moments;
// brute-force detailed balance for MH/MALA/HMC; HMC linear-map closed form; AIES affine
// invariance and the d=2 anisotropic-Gaussian variance test; covariance vs numpy.cov/LAPACK.
// PARITY UNPINNED by the paper (our own definitions, pinned only by finite differences /
// continuity): the box-penalty form and constants (reading R6), the jitter rule of the
// covariance update (R14).
//
// Section/equation/line references are to /root/reference/PAPER.md ("P:Lnn").

#include <cmath>
#include <cstdint>
#include <cstdlib>
#include <cstring>
#include <limits>
#include <vector>

#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

// ---------------------------------------------------------------------------------------------
// RNG: Philox4x32-10 (Salmon, Moraes, Dror, Shaw, SC'11).  north_star: "Philox counter-based RNG
// keyed by (seed, chain, step)"; stream layout = reading R1.
// ---------------------------------------------------------------------------------------------
void philox4x32_10(const uint32_t ctr_in[4], const uint32_t key_in[2], uint32_t out[4]) {
  uint32_t c0 = ctr_in[0], c1 = ctr_in[1], c2 = ctr_in[2], c3 = ctr_in[3];
  uint32_t k0 = key_in[0], k1 = key_in[1];
  for (int round = 0; round < 10; ++round) {
    const uint64_t p0 = (uint64_t)0xD2511F53u * (uint64_t)c0;
    const uint64_t p1 = (uint64_t)0xCD9E8D57u * (uint64_t)c2;
    const uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
    const uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
    const uint32_t n0 = hi1 ^ c1 ^ k0;
    const uint32_t n1 = lo1;
    const uint32_t n2 = hi0 ^ c3 ^ k1;
    const uint32_t n3 = lo0;
    c0 = n0; c1 = n1; c2 = n2; c3 = n3;
    k0 += 0x9E3779B9u;  // Weyl constants, bumped after every round
    k1 += 0xBB67AE85u;
  }
  out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

// counter = (chain, step lo32, step hi32, slot); key = (seed lo32, seed hi32)   [R1]
void philox_block(uint64_t seed, uint64_t chain, uint64_t step, uint32_t slot, uint32_t out[4]) {
  const uint32_t ctr[4] = {(uint32_t)chain, (uint32_t)step, (uint32_t)(step >> 32), slot};
  const uint32_t key[2] = {(uint32_t)seed, (uint32_t)(seed >> 32)};
  philox4x32_10(ctr, key, out);
}

// u = ((x >> 9) + 0.5) * 2^-23 in (0,1).  (2k+1) 2^-24 with k < 2^23 needs at most 24 mantissa
// bits, so u is exact in fp32 and in fp64 and never 0 or 1.   [R2; SURVEY's (x>>8) 2^-24 variant
// is NOT fp32-exact for x >= 2^31, so the 23-bit form is used]
double u01(uint32_t x) { return ((double)(x >> 9) + 0.5) * (1.0 / 8388608.0); }

// Box–Muller: r = sqrt(-2 ln u1), phi = 2 pi u2, (r cos phi, r sin phi)   [R3]
void box_muller(uint32_t w0, uint32_t w1, double* n0, double* n1) {
  const double u1 = u01(w0), u2 = u01(w1);
  const double r = std::sqrt(-2.0 * std::log(u1));
  const double phi = 2.0 * M_PI * u2;
  *n0 = r * std::cos(phi);
  *n1 = r * std::sin(phi);
}

// slot 1+j -> normals for dims 4j..4j+3: (w0,w1) -> dims 4j,4j+1; (w2,w3) -> 4j+2,4j+3   [R1]
void draw_normals(uint64_t seed, uint64_t chain, uint64_t step, int d, double* xi) {
  const int nblk = (d + 3) / 4;
  for (int j = 0; j < nblk; ++j) {
    uint32_t w[4];
    philox_block(seed, chain, step, (uint32_t)(1 + j), w);
    double n[4];
    box_muller(w[0], w[1], &n[0], &n[1]);
    box_muller(w[2], w[3], &n[2], &n[3]);
    for (int t = 0; t < 4; ++t)
      if (4 * j + t < d) xi[4 * j + t] = n[t];  // surplus normals discarded
  }
}

// slot 0 = control block: word0 -> accept uniform, word1 -> AIES u_z, word2 -> AIES partner raw
void draw_control(uint64_t seed, uint64_t chain, uint64_t step, double* u_acc, double* u_z,
                  uint32_t* partner_raw) {
  uint32_t w[4];
  philox_block(seed, chain, step, 0u, w);
  *u_acc = u01(w[0]);
  *u_z = u01(w[1]);
  *partner_raw = w[2];
}

// ---------------------------------------------------------------------------------------------
// Target   log pi(theta) = -1/2 (theta-mu)^T Sigma^-1 (theta-mu) + s*MLP(theta) + banana - pen
// (stand-in for the paper's emulator log_prob_fn)
// ---------------------------------------------------------------------------------------------
struct Oracle {
  int d = 0;
  int n_affine = 0;
  std::vector<int> widths;
  std::vector<std::vector<double>> W, b;  // promoted from the fp32 inputs
  int activation = 0;
  double mlp_scale = 0.0;
  bool has_gauss = false;
  std::vector<double> mu, P;  // P = Sigma^-1 (dense, used as given)
  bool has_box = false;
  std::vector<double> lo, hi;
  double pen_kappa = 1.0, pen_gamma = 100.0;
  int banana_i = -1, banana_j = -1;
  double banana_sigma = 0.1;
  std::vector<double> L;  // lower-triangular whitening factor, row-major d*d
  // SURVEY 8(f)#1 (a larger step for some parameters): per-dimension step factors s_i
  // in whitened space (reading R20) and the hard-box option (reading R21)
  std::vector<double> step_scale;  // [d], all 1 by default
  bool hard_box = false;
  // covariance adaptation (O6)
  int64_t adapt_every = 0;
  double jitter = 1e-6;
  int64_t win_steps = 0;
  double cov_n = 0.0;
  std::vector<double> cov_mean, cov_M2;
  int64_t n_updates = 0, n_update_failures = 0;
  // when chains are sharded over ranks, local chain c draws the Philox stream of the GLOBAL
  // chain id chain0 + c (counter word 0 of reading R1); 0 = the single-process stream
  uint64_t chain0 = 0;
};

double act_f(int kind, double a, double* dact) {
  if (kind == 0) {  // tanh; tanh' = 1 - h^2
    const double h = std::tanh(a);
    *dact = 1.0 - h * h;
    return h;
  }
  // SiLU(a) = a*sigma(a); SiLU' = sigma(a) (1 + a (1 - sigma(a))); sigma overflow-safe
  const double e = std::exp(-std::fabs(a));
  const double sg = (a >= 0.0) ? 1.0 / (1.0 + e) : e / (1.0 + e);
  *dact = sg * (1.0 + a * (1.0 - sg));
  return a * sg;
}

// A1b forward + A1c input-gradient (no weight gradients).  grad may be null.
double mlp_eval(const Oracle& o, const double* theta, double* grad) {
  const int K1 = o.n_affine;  // number of affine maps (K hidden + 1 output)
  std::vector<std::vector<double>> h(K1 + 1), dact(K1 + 1);
  h[0].assign(theta, theta + o.d);
  for (int k = 0; k < K1; ++k) {
    const int nin = o.widths[k], nout = o.widths[k + 1];
    h[k + 1].assign(nout, 0.0);
    dact[k + 1].assign(nout, 1.0);
    for (int r = 0; r < nout; ++r) {
      double a = o.b[k][r];
      for (int c = 0; c < nin; ++c) a += o.W[k][(size_t)r * nin + c] * h[k][c];
      if (k < K1 - 1) {
        double da;
        h[k + 1][r] = act_f(o.activation, a, &da);
        dact[k + 1][r] = da;
      } else {
        h[k + 1][r] = a;  // linear scalar output
      }
    }
  }
  const double out = h[K1][0];
  if (grad) {
    // delta_K1 = 1 (d out / d out); delta_{k} = (W_{k+1}^T delta_{k+1}) .* act'(a_k)
    std::vector<double> delta(1, 1.0);
    for (int k = K1 - 1; k >= 0; --k) {
      const int nin = o.widths[k], nout = o.widths[k + 1];
      std::vector<double> prev(nin, 0.0);
      for (int c = 0; c < nin; ++c) {
        double s = 0.0;
        for (int r = 0; r < nout; ++r) s += o.W[k][(size_t)r * nin + c] * delta[r];
        prev[c] = (k > 0) ? s * dact[k][c] : s;
      }
      delta.swap(prev);
    }
    for (int i = 0; i < o.d; ++i) grad[i] = delta[i];
  }
  return out;
}

// Reading R6 (paper: "smooth exponential penalty outside the domain ... preserving
// differentiability"; form and constants are ours):
//   t_i = gamma * max(0, lo_i - th_i, th_i - hi_i) / (hi_i - lo_i);  pen = kappa * sum_i f(t_i)
//   f(t) = e^t - 1 - t for t <= 40, continued linearly with slope e^40 - 1 beyond.
double pen_f(double t, double* df) {
  if (t <= 0.0) { *df = 0.0; return 0.0; }
  if (t <= 40.0) { *df = std::expm1(t); return std::expm1(t) - t; }
  const double s40 = std::expm1(40.0);
  *df = s40;
  return (s40 - 40.0) + s40 * (t - 40.0);
}

double target_eval(const Oracle& o, const double* theta, double* grad) {
  const int d = o.d;
  double logp = 0.0;
  if (grad) for (int i = 0; i < d; ++i) grad[i] = 0.0;
  if (o.has_gauss) {  // A1a, the plain definition with the dense precision matrix
    std::vector<double> r(d);
    for (int i = 0; i < d; ++i) r[i] = theta[i] - o.mu[i];
    double q = 0.0;
    for (int i = 0; i < d; ++i) {
      double v = 0.0, vt = 0.0;
      for (int j = 0; j < d; ++j) {
        v += o.P[(size_t)i * d + j] * r[j];
        vt += o.P[(size_t)j * d + i] * r[j];
      }
      q += r[i] * v;
      if (grad) grad[i] += -0.5 * (v + vt);
    }
    logp += -0.5 * q;
  }
  if (o.n_affine > 0 && o.mlp_scale != 0.0) {  // A1b / A1c
    std::vector<double> g(d);
    const double out = mlp_eval(o, theta, grad ? g.data() : nullptr);
    logp += o.mlp_scale * out;
    if (grad) for (int i = 0; i < d; ++i) grad[i] += o.mlp_scale * g[i];
  }
  if (o.banana_i >= 0) {  // A1d: -(th_j - th_i^2)^2 / (2 sigma^2)
    const double ti = theta[o.banana_i], tj = theta[o.banana_j];
    const double t = tj - ti * ti, s2 = o.banana_sigma * o.banana_sigma;
    logp += -t * t / (2.0 * s2);
    if (grad) {
      grad[o.banana_j] += -t / s2;
      grad[o.banana_i] += 2.0 * ti * t / s2;
    }
  }
  if (o.has_box && o.hard_box) {  // reading R21: log pi = -inf outside [lo, hi] (no penalty term)
    for (int i = 0; i < d; ++i)
      if (theta[i] < o.lo[i] || theta[i] > o.hi[i]) logp = -INFINITY;
  } else if (o.has_box) {  // A1e
    double pen = 0.0;
    for (int i = 0; i < d; ++i) {
      const double width = o.hi[i] - o.lo[i];
      double ex = 0.0, sgn = 0.0;
      if (theta[i] < o.lo[i]) { ex = o.lo[i] - theta[i]; sgn = -1.0; }
      else if (theta[i] > o.hi[i]) { ex = theta[i] - o.hi[i]; sgn = 1.0; }
      if (ex > 0.0) {
        double df;
        pen += pen_f(o.pen_gamma * ex / width, &df);
        if (grad) grad[i] -= o.pen_kappa * df * o.pen_gamma / width * sgn;
      }
    }
    logp -= o.pen_kappa * pen;
  }
  return logp;
}

// Whitening, eq (2.4)-(2.5) P:L78-80:  x = mu + L z.  State is held as theta, so a step
// delta z in whitened space is  theta' = theta + L dz  and  g_z = L^T grad_theta  (reading R12).
void L_apply(const Oracle& o, const double* dz, double* out) {  // out = L dz (lower triangular)
  for (int i = 0; i < o.d; ++i) {
    double s = 0.0;
    for (int j = 0; j <= i; ++j) s += o.L[(size_t)i * o.d + j] * dz[j];
    out[i] = s;
  }
}
void Lt_apply(const Oracle& o, const double* g, double* out) {  // out = L^T g
  for (int j = 0; j < o.d; ++j) {
    double s = 0.0;
    for (int i = j; i < o.d; ++i) s += o.L[(size_t)i * o.d + j] * g[i];
    out[j] = s;
  }
}

// Accept rule (reading R7): accept iff log u < log alpha; NaN -> reject; +inf -> accept.
bool accept_rule(double u, double log_alpha) { return std::log(u) < log_alpha; }

// ---------------------------------------------------------------------------------------------
// Deterministic single-step maps ("given the random numbers").  The step drivers below draw the
// random numbers and call these; the detailed-balance / closed-form pins call these directly.
// ---------------------------------------------------------------------------------------------

// Per-dimension steps (reading R20): coordinate i of the whitened space moves with eps_i = eps s_i in MH
// and in the HMC leap-frog (drift and kick); MALA, the one-step limit, has drift eps s_i^2 g_i and noise
// sqrt(2 eps) s_i xi_i, i.e. eq (2.3) with eps_i = eps s_i^2 and q(.|z) = N(z + E g_z, 2E), E = diag(eps_i).
// O2 MH (reading R5): theta' = theta + eps L xi; log alpha = logpi' - logpi
void mh_map(const Oracle& o, const double* theta, double logp, const double* xi, double eps,
            double* theta_p, double* logp_p, double* log_alpha) {
  const int d = o.d;
  std::vector<double> dz(d), dx(d);
  for (int i = 0; i < d; ++i) dz[i] = eps * o.step_scale[i] * xi[i];
  L_apply(o, dz.data(), dx.data());
  for (int i = 0; i < d; ++i) theta_p[i] = theta[i] + dx[i];
  *logp_p = target_eval(o, theta_p, nullptr);
  *log_alpha = *logp_p - logp;
}

// O3 MALA, eq (2.3) P:L70 in whitened space (reading R4: eps multiplies the gradient,
// sqrt(2 eps) the noise).  Proposal q(.|z) = N(z + eps g_z, 2 eps 1).
//   log alpha = logpi' - logpi + log q(z|z') - log q(z'|z)
//   log q(z'|z) = -|z' - z - eps g_z|^2/(4 eps) = -|sqrt(2eps) xi|^2/(4 eps)
//   log q(z|z') = -|z - z' - eps g_z'|^2/(4 eps) = -|eps (g_z + g_z') + sqrt(2eps) xi|^2/(4 eps)
void mala_map(const Oracle& o, const double* theta, double logp, const double* grad,
              const double* xi, double eps, double* theta_p, double* logp_p, double* grad_p,
              double* log_alpha) {
  const int d = o.d;
  std::vector<double> gz(d), dz(d), dx(d), gzp(d);
  Lt_apply(o, grad, gz.data());
  std::vector<double> ei(d), sq(d);
  for (int i = 0; i < d; ++i) {
    ei[i] = eps * o.step_scale[i] * o.step_scale[i];
    sq[i] = std::sqrt(2.0 * ei[i]);
  }
  for (int i = 0; i < d; ++i) dz[i] = ei[i] * gz[i] + sq[i] * xi[i];
  L_apply(o, dz.data(), dx.data());
  for (int i = 0; i < d; ++i) theta_p[i] = theta[i] + dx[i];
  *logp_p = target_eval(o, theta_p, grad_p);
  Lt_apply(o, grad_p, gzp.data());
  double fwd = 0.0, bwd = 0.0;
  for (int i = 0; i < d; ++i) {
    const double f = sq[i] * xi[i];                              // z' - z - eps_i g_z
    const double r = -(ei[i] * (gz[i] + gzp[i]) + sq[i] * xi[i]);  // z - z' - eps_i g_z'
    fwd += f * f / (4.0 * ei[i]);
    bwd += r * r / (4.0 * ei[i]);
  }
  *log_alpha = *logp_p - logp + (-bwd) - (-fwd);
}

// O4 HMC: Hamiltonian eq (2.1)/(2.8) P:L56, L96 with identity mass after whitening;
// leap-frog as kick-drift-kick (reading R13); log alpha = H0 - H1.
void hmc_map(const Oracle& o, const double* theta, double logp, const double* grad,
             const double* q0, double eps, int n_leapfrog, double* theta_p, double* logp_p,
             double* grad_p, double* q_p, double* log_alpha) {
  const int d = o.d;
  std::vector<double> q(q0, q0 + d), gz(d), dx(d), dz(d), th(theta, theta + d), g(grad, grad + d);
  double kin0 = 0.0;
  for (int i = 0; i < d; ++i) kin0 += q[i] * q[i];
  const double H0 = -logp + 0.5 * kin0;
  Lt_apply(o, g.data(), gz.data());
  const std::vector<double>& sc = o.step_scale;
  for (int i = 0; i < d; ++i) q[i] += 0.5 * eps * sc[i] * gz[i];  // half kick
  double lp = logp;
  for (int l = 1; l <= n_leapfrog; ++l) {
    for (int i = 0; i < d; ++i) dz[i] = eps * sc[i] * q[i];  // drift: z += eps q  <=>  theta += eps L q
    L_apply(o, dz.data(), dx.data());
    for (int i = 0; i < d; ++i) th[i] += dx[i];
    lp = target_eval(o, th.data(), g.data());
    Lt_apply(o, g.data(), gz.data());
    const double c = (l < n_leapfrog) ? eps : 0.5 * eps;  // full kick inside, half kick at the end
    for (int i = 0; i < d; ++i) q[i] += c * sc[i] * gz[i];
  }
  double kin1 = 0.0;
  for (int i = 0; i < d; ++i) kin1 += q[i] * q[i];
  const double H1 = -lp + 0.5 * kin1;
  for (int i = 0; i < d; ++i) { theta_p[i] = th[i]; grad_p[i] = g[i]; q_p[i] = q[i]; }
  *logp_p = lp;
  *log_alpha = H0 - H1;
}

// O5 AIES stretch move: eq (2.13); z from eq (2.15); acceptance factor z^(d-1)
// from Goodman & Weare (ref [13] P:L368; reading R9).  No whitening (footnote 2).
double stretch_z(double u, double a) { return (u * (a - 1.0) + 1.0) * (u * (a - 1.0) + 1.0) / a; }

void aies_map(const Oracle& o, const double* theta_i, double logp_i, const double* theta_j,
              double z, double* theta_p, double* logp_p, double* log_alpha) {
  const int d = o.d;
  for (int k = 0; k < d; ++k) theta_p[k] = theta_j[k] + z * (theta_i[k] - theta_j[k]);
  *logp_p = target_eval(o, theta_p, nullptr);
  *log_alpha = (double)(d - 1) * std::log(z) + *logp_p - logp_i;
}

// Differential-evolution move, eq (2.16) P:L170-176 (reading R23):
//   x_i' = x_i + gamma (x_j - x_k),  gamma = (1 + eta) 2.38 / sqrt(2 d),  eta ~ N(0, sigma_gamma).
// j and k are two DIFFERENT walkers; swapping them flips the displacement, so the proposal is symmetric
// and log alpha = log pi(x') - log pi(x_i) with no extra factor.
void de_map(const Oracle& o, const double* theta_i, double logp_i, const double* theta_j,
            const double* theta_k, double gamma, double* theta_p, double* logp_p, double* log_alpha) {
  const int d = o.d;
  for (int q = 0; q < d; ++q) theta_p[q] = theta_i[q] + gamma * (theta_j[q] - theta_k[q]);
  *logp_p = target_eval(o, theta_p, nullptr);
  *log_alpha = *logp_p - logp_i;
}

// ---------------------------------------------------------------------------------------------
// O6 covariance adaptation (reading R14)
// ---------------------------------------------------------------------------------------------
void cov_reset(Oracle& o) {
  o.win_steps = 0;
  o.cov_n = 0.0;
  o.cov_mean.assign(o.d, 0.0);
  o.cov_M2.assign((size_t)o.d * o.d, 0.0);
}

void cov_push(Oracle& o, const double* x) {  // Welford update with one sample
  const int d = o.d;
  o.cov_n += 1.0;
  std::vector<double> delta(d);
  for (int i = 0; i < d; ++i) {
    delta[i] = x[i] - o.cov_mean[i];
    o.cov_mean[i] += delta[i] / o.cov_n;
  }
  for (int i = 0; i < d; ++i)
    for (int j = 0; j < d; ++j)
      o.cov_M2[(size_t)i * d + j] += delta[i] * (x[j] - o.cov_mean[j]);
}

bool cholesky_lower(const std::vector<double>& C, int d, std::vector<double>& Lout) {
  Lout.assign((size_t)d * d, 0.0);
  for (int j = 0; j < d; ++j) {
    double s = C[(size_t)j * d + j];
    for (int k = 0; k < j; ++k) s -= Lout[(size_t)j * d + k] * Lout[(size_t)j * d + k];
    if (!(s > 0.0)) return false;
    const double ljj = std::sqrt(s);
    Lout[(size_t)j * d + j] = ljj;
    for (int i = j + 1; i < d; ++i) {
      double t = C[(size_t)i * d + j];
      for (int k = 0; k < j; ++k) t -= Lout[(size_t)i * d + k] * Lout[(size_t)j * d + k];
      Lout[(size_t)i * d + j] = t / ljj;
    }
  }
  return true;
}

// C = M2/(n-1); C += jitter*diag(C); L = chol(C); on failure jitter *= 10, up to 5 retries; else
// keep the old L.
void cov_update_whitening(Oracle& o) {
  const int d = o.d;
  if (o.cov_n >= 2.0) {
    std::vector<double> C((size_t)d * d), Ltry;
    double jit = o.jitter;
    bool ok = false;
    for (int attempt = 0; attempt < 6 && !ok; ++attempt) {
      for (int i = 0; i < d; ++i)
        for (int j = 0; j < d; ++j) {
          // symmetrised scatter / (n-1)
          C[(size_t)i * d + j] =
              0.5 * (o.cov_M2[(size_t)i * d + j] + o.cov_M2[(size_t)j * d + i]) / (o.cov_n - 1.0);
        }
      for (int i = 0; i < d; ++i) C[(size_t)i * d + i] *= (1.0 + jit);
      ok = cholesky_lower(C, d, Ltry);
      jit *= 10.0;
    }
    if (ok) { o.L = Ltry; o.n_updates++; } else { o.n_update_failures++; }
  } else {
    o.n_update_failures++;
  }
  cov_reset(o);
}

void adapt_after_step(Oracle& o, int64_t B, const double* theta) {
  if (o.adapt_every <= 0) return;
  for (int64_t c = 0; c < B; ++c) cov_push(o, theta + c * o.d);  // post-accept states, all chains
  o.win_steps++;
  if (o.win_steps >= o.adapt_every) cov_update_whitening(o);
}

void write_trace(const Oracle& o, double* trace, int thin, int64_t local_step, int64_t B,
                 const double* theta) {
  if (!trace || thin <= 0) return;
  if ((local_step + 1) % thin != 0) return;
  const int64_t slot = (local_step + 1) / thin - 1;
  std::memcpy(trace + (size_t)slot * B * o.d, theta, sizeof(double) * (size_t)B * o.d);
}

}  // namespace

// =============================================================================================
// C interface (host arrays only).  Mirrors include/best.h so one harness drives both.
// =============================================================================================
extern "C" {

struct oracle_config {
  int32_t d, n_affine;
  const int32_t* widths;   // [n_affine+1]
  const float* W_flat;     // W_1 .. W_{n_affine}, each row-major [widths[k+1]][widths[k]]
  const float* b_flat;     // b_1 .. b_{n_affine}
  int32_t activation;      // 0 tanh, 1 SiLU
  double mlp_scale;
  const double* mu;        // [d] or NULL
  const double* Sigma_inv; // [d*d] or NULL
  const double* lo;        // [d] or NULL
  const double* hi;
  double pen_kappa, pen_gamma;
  int32_t banana_i, banana_j;
  double banana_sigma;
  const double* L;         // [d*d] lower-triangular or NULL (identity)
};

void oracle_philox4x32_10(const uint32_t* ctr, const uint32_t* key, uint32_t* out) {
  philox4x32_10(ctr, key, out);
}
double oracle_u01(uint32_t x) { return u01(x); }
void oracle_normals(uint64_t seed, uint64_t chain, uint64_t step, int32_t d, double* xi) {
  draw_normals(seed, chain, step, d, xi);
}
void oracle_control(uint64_t seed, uint64_t chain, uint64_t step, double* u_acc, double* u_z,
                    uint32_t* partner_raw) {
  draw_control(seed, chain, step, u_acc, u_z, partner_raw);
}
double oracle_stretch_z(double u, double a) { return stretch_z(u, a); }
int32_t oracle_accept(double u, double log_alpha) { return accept_rule(u, log_alpha) ? 1 : 0; }
int32_t oracle_num_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

void* oracle_create(const oracle_config* c) {
  if (!c || c->d <= 0) return nullptr;
  Oracle* o = new Oracle();
  o->d = c->d;
  o->n_affine = c->n_affine;
  if (c->n_affine > 0) {
    o->widths.assign(c->widths, c->widths + c->n_affine + 1);
    size_t wo = 0, bo = 0;
    for (int k = 0; k < c->n_affine; ++k) {
      const size_t nin = o->widths[k], nout = o->widths[k + 1];
      o->W.emplace_back(c->W_flat + wo, c->W_flat + wo + nin * nout);
      o->b.emplace_back(c->b_flat + bo, c->b_flat + bo + nout);
      wo += nin * nout;
      bo += nout;
    }
  }
  o->activation = c->activation;
  o->mlp_scale = c->mlp_scale;
  if (c->mu && c->Sigma_inv) {
    o->has_gauss = true;
    o->mu.assign(c->mu, c->mu + c->d);
    o->P.assign(c->Sigma_inv, c->Sigma_inv + (size_t)c->d * c->d);
  }
  if (c->lo && c->hi) {
    o->has_box = true;
    o->lo.assign(c->lo, c->lo + c->d);
    o->hi.assign(c->hi, c->hi + c->d);
  }
  o->pen_kappa = c->pen_kappa;
  o->pen_gamma = c->pen_gamma;
  o->banana_i = c->banana_i;
  o->banana_j = c->banana_j;
  o->banana_sigma = c->banana_sigma;
  o->L.assign((size_t)c->d * c->d, 0.0);
  for (int i = 0; i < c->d; ++i)
    for (int j = 0; j <= i; ++j)
      o->L[(size_t)i * c->d + j] = c->L ? c->L[(size_t)i * c->d + j] : (i == j ? 1.0 : 0.0);
  o->step_scale.assign((size_t)c->d, 1.0);
  cov_reset(*o);
  return o;
}
// readings R20 / R21
void oracle_set_step_scale(void* h, const double* s) {
  Oracle& o = *static_cast<Oracle*>(h);
  for (int i = 0; i < o.d; ++i) o.step_scale[i] = s ? s[i] : 1.0;
}
void oracle_set_hard_box(void* h, int32_t on) { static_cast<Oracle*>(h)->hard_box = (on != 0); }
void oracle_destroy(void* h) { delete static_cast<Oracle*>(h); }

void oracle_set_whitening(void* h, const double* L) {
  Oracle& o = *static_cast<Oracle*>(h);
  for (int i = 0; i < o.d; ++i)
    for (int j = 0; j < o.d; ++j) o.L[(size_t)i * o.d + j] = (j <= i) ? L[(size_t)i * o.d + j] : 0.0;
}
void oracle_get_whitening(void* h, double* L) {
  Oracle& o = *static_cast<Oracle*>(h);
  std::memcpy(L, o.L.data(), sizeof(double) * (size_t)o.d * o.d);
}
// eq (2.12): the constant log|det L| = sum log diag(L)
double oracle_log_det_L(void* h) {
  Oracle& o = *static_cast<Oracle*>(h);
  double s = 0.0;
  for (int i = 0; i < o.d; ++i) s += std::log(o.L[(size_t)i * o.d + i]);
  return s;
}
void oracle_set_adaptation(void* h, int64_t adapt_every, double jitter) {
  Oracle& o = *static_cast<Oracle*>(h);
  o.adapt_every = adapt_every;
  o.jitter = jitter;
  cov_reset(o);
}
void oracle_adapt_stats(void* h, int64_t* n_updates, int64_t* n_failures) {
  Oracle& o = *static_cast<Oracle*>(h);
  *n_updates = o.n_updates;
  *n_failures = o.n_update_failures;
}
// covariance of an explicit sample set [n][d] through the same Welford/jitter/Cholesky code
int32_t oracle_cov_chol(void* h, const double* samples, int64_t n, double jitter, double* C_out,
                        double* L_out) {
  Oracle tmp;
  tmp.d = static_cast<Oracle*>(h)->d;
  tmp.jitter = jitter;
  tmp.L.assign((size_t)tmp.d * tmp.d, 0.0);
  cov_reset(tmp);
  for (int64_t r = 0; r < n; ++r) cov_push(tmp, samples + r * tmp.d);
  if (C_out)
    for (int i = 0; i < tmp.d * tmp.d; ++i) C_out[i] = tmp.cov_M2[i] / (tmp.cov_n - 1.0);
  cov_update_whitening(tmp);
  std::memcpy(L_out, tmp.L.data(), sizeof(double) * (size_t)tmp.d * tmp.d);
  return tmp.n_updates == 1 ? 0 : -1;
}

// log pi and gradient for n points, theta [n*d] (original space; reading: log|det L| NOT added)
void oracle_logp_grad(void* h, const double* theta, int64_t n, double* logp, double* grad) {
  const Oracle& o = *static_cast<Oracle*>(h);
#pragma omp parallel for schedule(dynamic, 1)
  for (int64_t c = 0; c < n; ++c)
    logp[c] = target_eval(o, theta + c * o.d, grad ? grad + c * o.d : nullptr);
}
void oracle_mlp(void* h, const double* theta, int64_t n, double* out, double* grad) {
  const Oracle& o = *static_cast<Oracle*>(h);
#pragma omp parallel for schedule(dynamic, 1)
  for (int64_t c = 0; c < n; ++c)
    out[c] = mlp_eval(o, theta + c * o.d, grad ? grad + c * o.d : nullptr);
}
double oracle_pen_f(double t, double* df) { return pen_f(t, df); }

// --- deterministic maps (random numbers supplied by the caller) -------------------------------
void oracle_mh_map(void* h, const double* theta, double logp, const double* xi, double eps,
                   double* theta_p, double* logp_p, double* log_alpha) {
  mh_map(*static_cast<Oracle*>(h), theta, logp, xi, eps, theta_p, logp_p, log_alpha);
}
void oracle_mala_map(void* h, const double* theta, double logp, const double* grad,
                     const double* xi, double eps, double* theta_p, double* logp_p, double* grad_p,
                     double* log_alpha) {
  mala_map(*static_cast<Oracle*>(h), theta, logp, grad, xi, eps, theta_p, logp_p, grad_p, log_alpha);
}
void oracle_hmc_map(void* h, const double* theta, double logp, const double* grad, const double* q0,
                    double eps, int32_t n_leapfrog, double* theta_p, double* logp_p, double* grad_p,
                    double* q_p, double* log_alpha) {
  hmc_map(*static_cast<Oracle*>(h), theta, logp, grad, q0, eps, n_leapfrog, theta_p, logp_p, grad_p,
          q_p, log_alpha);
}
void oracle_aies_map(void* h, const double* theta_i, double logp_i, const double* theta_j, double z,
                     double* theta_p, double* logp_p, double* log_alpha) {
  aies_map(*static_cast<Oracle*>(h), theta_i, logp_i, theta_j, z, theta_p, logp_p, log_alpha);
}

// --- step drivers ------------------------------------------------------------------------------
// State arrays are caller-owned: theta [B*d], logp [B], grad [B*d] (in/out), n_accept [B]
// (accumulated), last_log_alpha [B] (nullable, overwritten each step), trace [n/thin][B][d]
// (nullable).  `step0` is the global step counter of the first step of this call (the Philox
// `step`), so 1 x N steps == k x (N/k) steps bit-for-bit.

void oracle_set_chain_offset(void* h, uint64_t chain0) { static_cast<Oracle*>(h)->chain0 = chain0; }

void oracle_step_mh(void* h, int64_t B, double* theta, double* logp, uint64_t step0, int64_t n_steps,
                    uint64_t seed, double eps, uint64_t* n_accept, double* last_log_alpha,
                    double* trace, int32_t thin) {
  Oracle& o = *static_cast<Oracle*>(h);
  const int d = o.d;
  for (int64_t t = 0; t < n_steps; ++t) {
    const uint64_t step = step0 + (uint64_t)t;
#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t c = 0; c < B; ++c) {
      std::vector<double> xi(d), thp(d);
      double u, uz, lpp, la;
      uint32_t raw;
      draw_normals(seed, o.chain0 + (uint64_t)c, step, d, xi.data());
      draw_control(seed, o.chain0 + (uint64_t)c, step, &u, &uz, &raw);
      mh_map(o, theta + c * d, logp[c], xi.data(), eps, thp.data(), &lpp, &la);
      if (last_log_alpha) last_log_alpha[c] = la;
      if (accept_rule(u, la)) {
        std::memcpy(theta + c * d, thp.data(), sizeof(double) * d);
        logp[c] = lpp;
        n_accept[c] += 1;
      }
    }
    write_trace(o, trace, thin, t, B, theta);
    adapt_after_step(o, B, theta);
  }
}

void oracle_step_mala(void* h, int64_t B, double* theta, double* logp, double* grad, uint64_t step0,
                      int64_t n_steps, uint64_t seed, double eps, uint64_t* n_accept,
                      double* last_log_alpha, double* trace, int32_t thin) {
  Oracle& o = *static_cast<Oracle*>(h);
  const int d = o.d;
  for (int64_t t = 0; t < n_steps; ++t) {
    const uint64_t step = step0 + (uint64_t)t;
#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t c = 0; c < B; ++c) {
      std::vector<double> xi(d), thp(d), gp(d);
      double u, uz, lpp, la;
      uint32_t raw;
      draw_normals(seed, o.chain0 + (uint64_t)c, step, d, xi.data());
      draw_control(seed, o.chain0 + (uint64_t)c, step, &u, &uz, &raw);
      mala_map(o, theta + c * d, logp[c], grad + c * d, xi.data(), eps, thp.data(), &lpp, gp.data(),
               &la);
      if (last_log_alpha) last_log_alpha[c] = la;
      if (accept_rule(u, la)) {
        std::memcpy(theta + c * d, thp.data(), sizeof(double) * d);
        std::memcpy(grad + c * d, gp.data(), sizeof(double) * d);
        logp[c] = lpp;
        n_accept[c] += 1;
      }
    }
    write_trace(o, trace, thin, t, B, theta);
    adapt_after_step(o, B, theta);
  }
}

void oracle_step_hmc(void* h, int64_t B, double* theta, double* logp, double* grad, uint64_t step0,
                     int64_t n_traj, uint64_t seed, double eps, int32_t n_leapfrog,
                     uint64_t* n_accept, double* last_log_alpha, double* trace, int32_t thin) {
  Oracle& o = *static_cast<Oracle*>(h);
  const int d = o.d;
  for (int64_t t = 0; t < n_traj; ++t) {
    const uint64_t step = step0 + (uint64_t)t;  // Philox `step` = trajectory index (R1)
#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t c = 0; c < B; ++c) {
      std::vector<double> q(d), thp(d), gp(d), qp(d);
      double u, uz, lpp, la;
      uint32_t raw;
      draw_normals(seed, o.chain0 + (uint64_t)c, step, d, q.data());  // momentum q ~ N(0, 1)
      draw_control(seed, o.chain0 + (uint64_t)c, step, &u, &uz, &raw);
      hmc_map(o, theta + c * d, logp[c], grad + c * d, q.data(), eps, n_leapfrog, thp.data(), &lpp,
              gp.data(), qp.data(), &la);
      if (last_log_alpha) last_log_alpha[c] = la;
      if (accept_rule(u, la)) {
        std::memcpy(theta + c * d, thp.data(), sizeof(double) * d);
        std::memcpy(grad + c * d, gp.data(), sizeof(double) * d);
        logp[c] = lpp;
        n_accept[c] += 1;
      }
    }
    write_trace(o, trace, thin, t, B, theta);
    adapt_after_step(o, B, theta);
  }
}

// Halves S0 = [0,B/2), S1 = [B/2,B).  For h in (0,1): every i in S_h moves against the other
// half's CURRENT positions; S1 sees the updated S0 (reading R11).  partner j = other-half offset
// + floor(raw * (B/2) / 2^32)  (high word of a 32x32 multiply).
int32_t oracle_step_aies(void* h, int64_t B, double* theta, double* logp, uint64_t step0,
                         int64_t n_steps, uint64_t seed, double a, uint64_t* n_accept,
                         double* last_log_alpha, double* trace, int32_t thin) {
  Oracle& o = *static_cast<Oracle*>(h);
  const int d = o.d;
  if (B < 2 || (B % 2) != 0 || !(a > 1.0)) return -1;
  const int64_t half = B / 2;
  for (int64_t t = 0; t < n_steps; ++t) {
    const uint64_t step = step0 + (uint64_t)t;
    for (int hh = 0; hh < 2; ++hh) {
      const int64_t own0 = hh == 0 ? 0 : half, other0 = hh == 0 ? half : 0;
      std::vector<double> newth((size_t)half * d), newlp(half);
      std::vector<uint8_t> acc(half);
#pragma omp parallel for schedule(dynamic, 1)
      for (int64_t r = 0; r < half; ++r) {
        const int64_t i = own0 + r;
        double u, uz, lpp, la;
        uint32_t raw;
        draw_control(seed, o.chain0 + (uint64_t)i, step, &u, &uz, &raw);
        const int64_t j = other0 + (int64_t)(((uint64_t)raw * (uint64_t)half) >> 32);
        const double z = stretch_z(uz, a);
        aies_map(o, theta + i * d, logp[i], theta + j * d, z, newth.data() + r * d, &lpp, &la);
        newlp[r] = lpp;
        if (last_log_alpha) last_log_alpha[i] = la;
        acc[r] = accept_rule(u, la) ? 1 : 0;
      }
      for (int64_t r = 0; r < half; ++r)
        if (acc[r]) {
          const int64_t i = own0 + r;
          std::memcpy(theta + i * d, newth.data() + r * d, sizeof(double) * d);
          logp[i] = newlp[r];
          n_accept[i] += 1;
        }
    }
    write_trace(o, trace, thin, t, B, theta);
  }
  return 0;
}

// DE move with the ensemble split of R11 (reading R23): every i in half S_h draws j != k uniformly from
// the OTHER half's current positions.  From the control block (slot 0): word0 -> accept uniform,
// word2 -> j = other0 + floor(w2 (B/2) / 2^32), word3 -> k' = floor(w3 (B/2 - 1) / 2^32), k = other0 + k'
// + (k' >= j - other0) (uniform over the B/2 - 1 walkers that are not j); eta = sigma_gamma * (first normal
// of slot 1).
void oracle_de_map(void* h, const double* theta_i, double logp_i, const double* theta_j,
                   const double* theta_k, double gamma, double* theta_p, double* logp_p, double* log_alpha) {
  de_map(*static_cast<Oracle*>(h), theta_i, logp_i, theta_j, theta_k, gamma, theta_p, logp_p, log_alpha);
}
int32_t oracle_step_aies_de(void* h, int64_t B, double* theta, double* logp, uint64_t step0,
                            int64_t n_steps, uint64_t seed, double sigma_gamma, uint64_t* n_accept,
                            double* last_log_alpha, double* trace, int32_t thin) {
  Oracle& o = *static_cast<Oracle*>(h);
  const int d = o.d;
  if (B < 4 || (B % 2) != 0 || !(sigma_gamma >= 0.0)) return -1;
  const int64_t half = B / 2;
  const double gamma0 = 2.38 / std::sqrt(2.0 * (double)d);
  for (int64_t t = 0; t < n_steps; ++t) {
    const uint64_t step = step0 + (uint64_t)t;
    for (int hh = 0; hh < 2; ++hh) {
      const int64_t own0 = hh == 0 ? 0 : half, other0 = hh == 0 ? half : 0;
      std::vector<double> newth((size_t)half * d), newlp(half);
      std::vector<uint8_t> acc(half);
#pragma omp parallel for schedule(dynamic, 1)
      for (int64_t r = 0; r < half; ++r) {
        const int64_t i = own0 + r;
        uint32_t w[4];
        philox_block(seed, o.chain0 + (uint64_t)i, step, 0u, w);
        const double u = u01(w[0]);
        const int64_t jr = (int64_t)(((uint64_t)w[2] * (uint64_t)half) >> 32);
        int64_t kr = (int64_t)(((uint64_t)w[3] * (uint64_t)(half - 1)) >> 32);
        if (kr >= jr) kr += 1;
        std::vector<double> xi(4 * ((d + 3) / 4));
        draw_normals(seed, o.chain0 + (uint64_t)i, step, d, xi.data());
        const double gamma = (1.0 + sigma_gamma * xi[0]) * gamma0;
        double lpp, la;
        de_map(o, theta + i * d, logp[i], theta + (other0 + jr) * d, theta + (other0 + kr) * d, gamma,
               newth.data() + r * d, &lpp, &la);
        newlp[r] = lpp;
        if (last_log_alpha) last_log_alpha[i] = la;
        acc[r] = accept_rule(u, la) ? 1 : 0;
      }
      for (int64_t r = 0; r < half; ++r)
        if (acc[r]) {
          const int64_t i = own0 + r;
          std::memcpy(theta + i * d, newth.data() + r * d, sizeof(double) * d);
          logp[i] = newlp[r];
          n_accept[i] += 1;
        }
    }
    write_trace(o, trace, thin, t, B, theta);
  }
  return 0;
}

}  // extern "C"
