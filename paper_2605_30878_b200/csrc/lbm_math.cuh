// lbm_math.cuh — node-local arithmetic of the color-gradient D2Q9 update (device code, fp64/fp32).
//
// Written from PAPER.md (App. A, Eq. A1-A15; §II Eq. 4); shares nothing with oracle/.
// Differences from the paper's matrix form, all exact rewrites:
//   * Populations are held as deviations n_i = N_i - chi_i (Eq. A7 color weights).  Every moment
//     the update needs (sum_{i!=0} N_i, j, Pi_xx - Pi_yy, Pi_xy) is linear in N and the chi-part
//     is known in closed form, so the deviation form is exact and keeps fp32 usable at density
//     ratio 1000 where p ~ 1e-7 sits on top of chi_0 ~ 0.93.
//   * Because S = diag(1,1,1,1,1,1,1,s,s) (Eq. A3, :271) and the forcing populations F_i (A8)
//     have zero second moments, Eq. A1 reduces to
//        N_i* = N_i^eq + (1-s)/4 [ (m7 - m7^eq) M_7i + (m8 - m8^eq) M_8i ] + F_i / 2
//     with M_7 = c_x^2 - c_y^2, M_8 = c_x c_y rows of Eq. A2 (|M_7|^2 = |M_8|^2 = 4).
//   * tau = 1/2 + 3 nu, nu = 1/D, D = phi/nu_l + (1-phi)/nu_g (:43, :273), so with r = 1/(D/2 + 3):
//        s = 1/tau = D r,  1 - s = (3 - D/2) r,  (tau - 1/2)/tau = 3 r.
#pragma once
#include <cuda_runtime.h>

namespace lbm {

// constants of one simulation in the device precision
template <typename R>
struct Consts {
  int nx, ny;
  size_t ps;            // element stride between population planes (>= nx*ny, padded so that the
                        // 18 plane streams of a step do not alias in the L2 sets)
  R rho_g, drho;        // rho = rho_g + drho * phi                              (:43)
  R inu_g, dinu;        // D = 1/nu = inu_g + dinu * phi                         (:43)
  R s48W, s15W;         // sigma*48/W and sigma*3W/2 of Eq. 4                    (:45)
  R twoW;               // 2/W of Eq. A12                                        (:307)
  R gbx, gby;           // body acceleration                                     (:39)
  R chi0, chi1, chi5;   // alpha, (1-alpha)/5, (1-alpha)/20                      (:285)
  R E, eps;             // e^eps and eps = -(4/W) cos(theta) of Eq. 9           (:78-80)
  R phi_solid;          // (1 + cos theta)/2                                     (:100)
  int ghost_rule;
  int all_links;        // INPLACE schedule at odd times: every population a node pulls sits in the node's own opposite
                        // slot, which is what the readers do for a bounce-back link
};

__device__ __forceinline__ double rcp_(double x) { return 1.0 / x; }
__device__ __forceinline__ float rcp_(float x) { return 1.0f / x; }
// 1/sqrt(x) for x > 0, else 0 (R16: the anti-diffusion term is dropped where grad phi vanishes)
__device__ __forceinline__ double rsqrt0_(double x) { return x > 0.0 ? rsqrt(x) : 0.0; }
__device__ __forceinline__ float rsqrt0_(float x) { return x > 0.0f ? rsqrtf(x) : 0.0f; }

// ---- two fp32 nodes in one 64-bit register pair: sm_100 packed FFMA2 / FADD2 / FMUL2 ----
struct F2 {
  float2 v;
};
__device__ __forceinline__ F2 f2(float a, float b) { return {make_float2(a, b)}; }
__device__ __forceinline__ F2 f2(float a) { return {make_float2(a, a)}; }
__device__ __forceinline__ F2 operator+(F2 a, F2 b) { return {__fadd2_rn(a.v, b.v)}; }
__device__ __forceinline__ F2 operator-(F2 a, F2 b) { return {__fadd2_rn(a.v, make_float2(-b.v.x, -b.v.y))}; }
__device__ __forceinline__ F2 operator*(F2 a, F2 b) { return {__fmul2_rn(a.v, b.v)}; }
__device__ __forceinline__ F2 operator-(F2 a) { return {make_float2(-a.v.x, -a.v.y)}; }
__device__ __forceinline__ F2 operator+(F2 a, float b) { return a + f2(b); }
__device__ __forceinline__ F2 operator+(float a, F2 b) { return f2(a) + b; }
__device__ __forceinline__ F2 operator-(F2 a, float b) { return a + f2(-b); }
__device__ __forceinline__ F2 operator-(float a, F2 b) { return f2(a) - b; }
__device__ __forceinline__ F2 operator*(F2 a, float b) { return a * f2(b); }
__device__ __forceinline__ F2 operator*(float a, F2 b) { return f2(a) * b; }
__device__ __forceinline__ float rcp_approx(float x) {
  float y;
  asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}
__device__ __forceinline__ float rsqrt_approx(float x) {
  float y;
  asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}
// arguments are O(1) normal numbers (rho >= rho_g, D/2 + 3 > 3): one MUFU each, ~1 ulp
__device__ __forceinline__ F2 rcp_(F2 a) { return f2(rcp_approx(a.v.x), rcp_approx(a.v.y)); }
// |grad phi|^2 below FLT_MIN counts as zero (R16): rsqrt.approx.ftz would flush it and return inf;
// the term it scales is O(phi (1 - phi)) ~ W |grad phi| / 4 < 1e-19 there
__device__ __forceinline__ F2 rsqrt0_(F2 a) {
  return f2(a.v.x >= 1.17549435e-38f ? rsqrt_approx(a.v.x) : 0.0f,
            a.v.y >= 1.17549435e-38f ? rsqrt_approx(a.v.y) : 0.0f);
}

template <typename R>
struct NodeOut {
  R rho, tau, ux, uy, p, Fx, Fy, gnorm;
};

// One fluid node.  n[q]: deviations of the post-stream populations; ph[q] = phi(x + c_q).
// Writes the post-collision deviations ns[q] = N_q* - chi_q and the full B_q* (Eq. A12).
// T is the value type: R itself (one node) or F2 (two nodes packed in one f32x2 register pair,
// FFMA2/FADD2/FMUL2).  MASKED: bmask (0 or 1 per node) zeroes every B_q* of a node that is not
// fluid (its packed partner is); all inputs must be finite.
template <typename T, typename R, bool WANT_B, bool MASKED>
__device__ __forceinline__ void node_update_t(const Consts<R>& C, const T (&n)[9], const T (&ph)[9],
                                              T (&ns)[9], T (&bs)[9], NodeOut<T>* out, T bmask) {
  const T phi = ph[0];
  // isotropic D2Q9 stencils (R8): grad = 3 sum w_i c_i phi(x+c_i), lap = 6 sum w_i (phi_i - phi_0)
  const T dax = ph[1] - ph[3], day = ph[2] - ph[4];
  const T gx = R(1.0 / 3.0) * dax + R(1.0 / 12.0) * ((ph[5] - ph[6]) + (ph[8] - ph[7]));
  const T gy = R(1.0 / 3.0) * day + R(1.0 / 12.0) * ((ph[5] - ph[8]) + (ph[6] - ph[7]));
  const T lap = R(2.0 / 3.0) * ((ph[1] + ph[3]) + (ph[2] + ph[4])) +
                R(1.0 / 6.0) * ((ph[5] + ph[7]) + (ph[6] + ph[8])) - R(10.0 / 3.0) * phi;

  // mixture rules (:43) and relaxation rate (:273)
  const T rho = C.rho_g + C.drho * phi;
  const T drx = C.drho * gx, dry = C.drho * gy;
  const T D = C.inu_g + C.dinu * phi;
  const T r = rcp_(R(0.5) * D + R(3.0));
  const T oms = (R(3.0) - R(0.5) * D) * r;   // 1 - 1/tau
  const T cv = R(-3.0) * r;                  // -(tau - 1/2)/tau
  const T irho = rcp_(rho);
  const T h = R(0.5) * irho;

  // surface tension force, Eq. 4 (:45); body force rho g (:39)
  const T omp = R(1.0) - phi;
  const T mu = -(C.s48W * (phi * omp) * (phi - R(0.5)) + C.s15W * lap);
  const T F0x = mu * gx + rho * C.gbx, F0y = mu * gy + rho * C.gby;

  // raw moments (deviation form; the chi-parts of j, m7, m8 vanish by symmetry)
  const T jx = (n[1] - n[3]) + ((n[5] - n[6]) + (n[8] - n[7]));
  const T jy = (n[2] - n[4]) + ((n[5] - n[8]) + (n[6] - n[7]));
  const T m7 = (n[1] + n[3]) - (n[2] + n[4]);
  const T m8 = (n[5] + n[7]) - (n[6] + n[8]);
  const T Sp = ((n[1] + n[3]) + (n[2] + n[4])) + ((n[5] + n[7]) + (n[6] + n[8]));

  // one Picard pass for the implicit (u, p, F_p, F_visc) coupling (R9, R10); A14 (:313), A15 (:315)
  // in deviation form: p = [c_s^2 sum_{i!=0} n_i - (w_0/2) u^2] / (1 - w_0) = 0.6 Sp - 0.4 u^2
  const T u0x = jx + F0x * h, u0y = jy + F0y * h;
  const T p0 = R(0.6) * Sp - R(0.4) * (u0x * u0x + u0y * u0y);
  const T m7n = m7 - (u0x * u0x - u0y * u0y);
  const T m8n = m8 - u0x * u0y;
  const T Fx = F0x - p0 * drx + cv * (R(0.5) * m7n * drx + m8n * dry);   // A9-A11 (:294-302)
  const T Fy = F0y - p0 * dry + cv * (m8n * drx - R(0.5) * m7n * dry);
  const T ux = jx + Fx * h, uy = jy + Fy * h;
  const T u2 = ux * ux + uy * uy;
  const T p = R(0.6) * Sp - R(0.4) * u2;

  // equilibrium A4 (:275) in deviation form, forcing A8 (:290), closed-form collision (see top)
  const T a7 = R(0.25) * oms * (m7 - (ux * ux - uy * uy));
  const T a8 = R(0.25) * oms * (m8 - ux * uy);
  const T ax = Fx * irho, ay = Fy * irho;            // F dt / rho
  const T base = R(3.0) * p - R(1.5) * u2;
  // axis directions: w = 1/9; cu = +-ux or +-uy; F_i/2 = (3 w /2) (a . c)
  const T ex = R(1.0 / 9.0) * (base + R(4.5) * ux * ux), ey = R(1.0 / 9.0) * (base + R(4.5) * uy * uy);
  const T lx = R(1.0 / 3.0) * ux + R(1.0 / 6.0) * ax, ly = R(1.0 / 3.0) * uy + R(1.0 / 6.0) * ay;
  ns[0] = R(-5.0 / 3.0) * p - R(2.0 / 3.0) * u2;
  ns[1] = ex + lx + a7;
  ns[3] = ex - lx + a7;
  ns[2] = ey + ly - a7;
  ns[4] = ey - ly - a7;
  // diagonals: w = 1/36; c = (+-1, +-1)
  const T upl = ux + uy, umi = ux - uy;
  const T epl = R(1.0 / 36.0) * (base + R(4.5) * upl * upl), emi = R(1.0 / 36.0) * (base + R(4.5) * umi * umi);
  const T lpl = R(1.0 / 12.0) * upl + R(1.0 / 24.0) * (ax + ay);
  const T lmi = R(1.0 / 12.0) * umi + R(1.0 / 24.0) * (ax - ay);
  ns[5] = epl + lpl + a8;
  ns[7] = epl - lpl + a8;
  ns[8] = emi + lmi - a8;
  ns[6] = emi - lmi - a8;

  const T g2 = gx * gx + gy * gy;
  if (WANT_B) {
    // segregation A12 (:307): B_i* = phi N_i* + (2/W)(c_i . n_phi) phi (1-phi) N_i^{eq,u=0}(p),
    // n_phi = grad phi/|grad phi| (term dropped where the gradient vanishes, R16)
    const T ig = rsqrt0_(g2);
    const T phb = MASKED ? phi * bmask : phi;
    const T kap = C.twoW * (phb * omp) * ig;
    const T kx = kap * gx, ky = kap * gy;
    const T q1 = C.chi1 + R(1.0 / 3.0) * p;      // N_i^{eq,u=0} = chi_i + 3 w_i p, axis
    const T q5 = C.chi5 + R(1.0 / 12.0) * p;     // diagonal
    bs[0] = phb * (C.chi0 + ns[0]);
    bs[1] = phb * (C.chi1 + ns[1]) + kx * q1;
    bs[3] = phb * (C.chi1 + ns[3]) - kx * q1;
    bs[2] = phb * (C.chi1 + ns[2]) + ky * q1;
    bs[4] = phb * (C.chi1 + ns[4]) - ky * q1;
    bs[5] = phb * (C.chi5 + ns[5]) + (kx + ky) * q5;
    bs[7] = phb * (C.chi5 + ns[7]) - (kx + ky) * q5;
    bs[8] = phb * (C.chi5 + ns[8]) + (kx - ky) * q5;
    bs[6] = phb * (C.chi5 + ns[6]) - (kx - ky) * q5;
  }
  if (out) {
    out->rho = rho;
    out->tau = R(0.5) + R(3.0) * rcp_(D);
    out->ux = ux; out->uy = uy; out->p = p; out->Fx = Fx; out->Fy = Fy;
    out->gnorm = g2 * rsqrt0_(g2);
  }
}

// one node, scalar arithmetic
template <typename R, bool WANT_B>
__device__ __forceinline__ void node_update(const Consts<R>& C, const R (&n)[9], const R (&ph)[9],
                                            R (&ns)[9], R (&bs)[9], NodeOut<R>* out) {
  node_update_t<R, R, WANT_B, false>(C, n, ph, ns, bs, out, R(1));
}

// Ghost-node rule.  rule 0: Eq. 9 (:78), phi_G = phi_F / (phi_F + (1 - phi_F) e^eps).
// rule 1: Eq. 10 (:84), phi_G = (2/eps)(a - s) - phi_F with a = 1 + eps/2, s = sqrt(a^2 - 2 eps phi_F), written as
// 4 phi_F/(a + s) - phi_F: the same value without the cancellation that makes the printed form 0/0 at
// theta = 90 deg (:87) and useless in fp32 near it.
template <typename R>
__device__ __forceinline__ R ghost_rule(const Consts<R>& C, R phiF) {
  if (C.ghost_rule == 0) return phiF / (phiF + (R(1.0) - phiF) * C.E);
  const R eps = C.eps;
  const R a = R(1.0) + R(0.5) * eps;
  return R(4.0) * phiF / (a + (R)sqrt((double)(a * a - R(2.0) * eps * phiF))) - phiF;
}

}  // namespace lbm
