// mf_event.cuh -- one event, S1 -> S8 (PAPER.md:59 pipeline), for the four processes of
// BASELINE.json configs 0-3 and the quark channel (process 4).  Returns F = w*f (pb), the weight
// before the 1/N (reading O8):
//   config 0   : F = J_V |M|^2 (1/(8 pi)) K / (2 s)
//   configs 1-3: F = J_V J_x f_g(x1) f_g(x2) |M|^2 S_f W_0 W_m Theta_cuts K / (2 shat)
//   process 4  : F = J_V J_x sum_q [f_q(x1) f_q~(x2) + f_q~(x1) f_q(x2)] |M|^2 W_0 W_m K / (2 shat)
#pragma once
#include "mf_device.cuh"
#include "generated/mf_me2_ee_mumu.cuh"
#include "generated/mf_me2_gg_tt.cuh"
#include "generated/mf_me2_gg_ttg.cuh"
#include "generated/mf_me2_gg_ttgg_lanes.cuh"     // gg -> tt~gg: one event over four lanes (gen/lanes.py)
#include "generated/mf_me2_qq_ttg.cuh"            // q q~ -> t t~ g and q g -> t t~ q (gen/quarks.py)
#include "generated/mf_me2_qg_ttq.cuh"

template <int PROC> struct MfProc;
// GROUP: threads that share the barrier points of the generated |M|^2 code (mf_device.cuh)
template <> struct MfProc<0> { static const int D = 2, N = 2, NGL = 0, GROUP = 128; };
template <> struct MfProc<1> { static const int D = 4, N = 2, NGL = 0, GROUP = 128; };
template <> struct MfProc<2> { static const int D = 7, N = 3, NGL = 1, GROUP = 128; };
#ifndef MF_TTGG_GROUP
#define MF_TTGG_GROUP 128     // gg -> tt~gg: 128-thread groups like gg -> tt~g (256 = the whole CTA shares the barrier points; tuning hook)
#endif
template <> struct MfProc<3> { static const int D = 10, N = 4, NGL = 2, GROUP = MF_TTGG_GROUP; };
// q q~ -> t t~ summed over five flavours: kinematics of process 1, PDF = flavour grid in global memory
template <> struct MfProc<4> { static const int D = 4, N = 2, NGL = 0, GROUP = 128; };
// p p -> t t~ at LO: the subprocesses g g -> t t~ and q q~ -> t t~ in one integrand (kinematics of process 1)
template <> struct MfProc<5> { static const int D = 4, N = 2, NGL = 0, GROUP = 128; };
// p p -> t t~ g through q q~ -> t t~ g (both beam orientations), and p p -> t t~ + quark jet through q g, g q, q~ g, g q~ ->
// t t~ q: kinematics, cuts (on the third final particle) and VEGAS dimensions of process 2, flavour grid
template <> struct MfProc<6> { static const int D = 7, N = 3, NGL = 1, GROUP = 128; };
template <> struct MfProc<7> { static const int D = 7, N = 3, NGL = 1, GROUP = 128; };
template <int PROC> struct MfPdf { static const bool FLAVOURS = PROC >= 4; };
// processes whose |M|^2 stage is heavy enough for the staged iteration path (front end / |M|^2 / reductions as three kernels)
template <int PROC> struct MfHeavy { static const bool value = PROC == 2 || PROC == 3; };
// partonic channels summed in one event (luminosity-weighted |M|^2): 1, or 2 (process 5: gg + qq~; process 6: q q~ and q~ q),
// or 4 (process 7: q g, g q, q~ g, g q~)
template <int PROC> struct MfChannels { static const int value = PROC == 7 ? 4 : (PROC == 5 || PROC == 6) ? 2 : 1; };
#define MF_NLUM 4
// Generator selection of the front end, template parameter CL:
//   0  the generators of the configs, nothing selectable (the path bench.py times: no branch)
//   1  classic 4n-random RAMBO, d = 2 + 4n; the tau map (O3 or O3') is a run-time, grid-uniform branch on P.gen
//   2  sequential RAMBO of the configs with the run-time branch on the tau map
template <int PROC, int CL> struct MfDim { static const int D = CL == 1 ? 2 + 4 * MfProc<PROC>::N : MfProc<PROC>::D; };
// bins are packed 6 bits each, 10 per 64-bit word: the second word holds dimensions 10.. of the classic generator
#define MF_PACK_DIMS 10
template <int D>
MF_HD void mf_pack_bins(const int bin[D], unsigned long long& lo, unsigned long long& hi) {
  lo = 0; hi = 0;
#pragma unroll
  for (int j = 0; j < D; ++j) {
    if (j < MF_PACK_DIMS) lo |= (unsigned long long)bin[j] << (6 * j);
    else hi |= (unsigned long long)bin[j] << (6 * (j - MF_PACK_DIMS));
  }
}

// optional per-event record (mf_integrand_eval's debug outputs)
struct MfEventRec {
  double y[MF_DMAX];
  double mom[6][4];
  double me2, pdf[2];
  int pass;
};

// inputs of the generated gg -> t t~ + gluons code: [E, mt, p3, p4, t-ingredients, t~-ingredients,
// then for every final gluon: k, polarisation ingredients] (order fixed by gen/amplitudes.py)
template <int N, typename T>
MF_HD void mf_me_inputs_gg(T rts, T mt, const T k[N][4], T* in) {
  in[0] = T(0.5) * rts; in[1] = mt;
#pragma unroll
  for (int c = 0; c < 4; ++c) { in[2 + c] = k[0][c]; in[6 + c] = k[1][c]; }
  mf_fermion_ing<T>(k[0], mt, in + 10);
  mf_fermion_ing<T>(k[1], mt, in + 15);
#pragma unroll
  for (int g = 2; g < N; ++g) {
#pragma unroll
    for (int c = 0; c < 4; ++c) in[20 + 9 * (g - 2) + c] = k[g][c];
    mf_gluon_ing<T>(k[g], in + 24 + 9 * (g - 2));
  }
}

// |M|^2 (averaged/summed, before the symmetry factor) in the real type T: double, or float for the fp32
// variant of the |M|^2 stage (A24: the front end and the reductions stay in fp64)
template <int PROC, typename T = double>
MF_HD T mf_me2(const MfParams& P, T rts, const T k[MfProc<PROC>::N][4]) {
  if (PROC == 0) {
    static_assert(MF_ME2_EE_MUMU_NIN == 20, "generator input layout changed");
    T in[20];
    const T E = T(0.5) * rts;
    const T pa[4] = {E, T(0.0), T(0.0), E}, pb[4] = {E, T(0.0), T(0.0), -E};
    mf_fermion_ing<T>(pa, T(0.0), in); mf_fermion_ing<T>(pb, T(0.0), in + 5);
    mf_fermion_ing<T>(k[0], T(0.0), in + 10); mf_fermion_ing<T>(k[1], T(0.0), in + 15);
    return T(P.me_pref) * mf_me2_ee_mumu<T>(in) / (rts * rts * rts * rts);      // e^4/4 * sum |L.R|^2 / s^2
  } else if (PROC == 4) {
    // O6q: the two-current contraction sum_hel |[vbar(pb) gamma^mu u(pa)][ubar(k1) gamma_mu v(k2)]|^2 of the generated
    // e+e- -> mu+mu- code, with massive outgoing spinors; me_pref = g_s^4 (2/9) / 4 (colour sum 2, 9 colours, 4 spins)
    T in[20];
    const T E = T(0.5) * rts;
    const T pa[4] = {E, T(0.0), T(0.0), E}, pb[4] = {E, T(0.0), T(0.0), -E};
    mf_fermion_ing<T>(pa, T(0.0), in); mf_fermion_ing<T>(pb, T(0.0), in + 5);
    mf_fermion_ing<T>(k[0], T(P.m_top), in + 10); mf_fermion_ing<T>(k[1], T(P.m_top), in + 15);
    return T(P.me_pref_qq) * mf_me2_ee_mumu<T>(in) / (rts * rts * rts * rts);
  } else if (PROC == 1) {
    static_assert(MF_ME2_GG_TT_NIN == 20, "generator input layout changed");
    T in[20];
    mf_me_inputs_gg<2, T>(rts, T(P.m_top), (const T(*)[4])k, in);
    return T(P.me_pref) * mf_me2_gg_tt<T>(in);
  } else if (PROC == 2) {
    static_assert(MF_ME2_GG_TTG_NIN == 29, "generator input layout changed");
    T in[29];
    mf_me_inputs_gg<3, T>(rts, T(P.m_top), (const T(*)[4])k, in);
    return T(P.me_pref) * mf_me2_gg_ttg<T>(in);
  } else {
    static_assert(PROC != 3 && PROC < 6, "gg -> tt~gg: mf_me2_ttgg_group (four lanes per event); processes 6, 7: mf_me2_2q");
    return T(0.0);
  }
}

// gg -> t t~ g with the loop-entering values of the helicity loop in shared memory (W: the thread's column of a [slot][S] tile)
#if defined(__CUDACC__)
template <typename T, int S>
__device__ __forceinline__ T mf_me2_ttg_smem(const MfParams& P, T rts, const T k[3][4], T* W) {
  static_assert(MF_ME2_GG_TTG_NIN == 29 && MF_ME2_GG_TTG_S_SCALE == MF_ME2_GG_TTG_SCALE, "generator input layout changed");
  {
    T in[29];
    mf_me_inputs_gg<3, T>(rts, T(P.m_top), k, in);
#pragma unroll
    for (int i = 0; i < 29; ++i) W[i * S] = in[i];
  }
  return T(P.me_pref) * mf_me2_gg_ttg_s<T, S>(W);
}
#endif

// ---- gg -> t t~ g g: one event over FOUR LANES (gen/lanes.py) -----------------------------------
// The four lanes of a group (lane & 3 = 0..3 of consecutive lanes) hold the same event (rts, k).  Lane l takes the
// six colour orderings that end with gluon l and runs the generated per-lane code on cyclically relabelled gluons
// (local label i = global gluon (i + l) mod 4); gluon currents and partial amplitudes are exchanged through the
// warp's shared-memory tile.  Global gluons: 0, 1 incoming along +z / -z, 2, 3 = k[2], k[3]; all-incoming momenta.
// tile: MF_LANES_TILE doubles per warp = the exchange slots X[slot][32], the parked loop invariants V[slot][32], and per
// event (8 per warp, stride MF_LANES_EVT: odd, so that the events fall on different banks) the table the generated code
// reads: mt, p4, spinor ingredients of t and t~, all-incoming momenta [4][4] and unit polarisation vectors [4][eps1, eps2]
// of the global gluons.  Every lane of the warp must call (warp barriers inside); returns |M|^2 on all four lanes of the group.
#if defined(__CUDACC__)
#define MF_LANES_EVT (MF_ME2_GG_TTGG_LANES_NEV + 24 + 2)
#define MF_LANES_TILE ((MF_ME2_GG_TTGG_LANES_SLOTS + MF_ME2_GG_TTGG_LANES_NV) * 32 + 8 * MF_LANES_EVT)
template <typename T>
__device__ __forceinline__ T mf_me2_ttgg_group(const MfParams& P, T rts, const T k[4][4], T* tile) {
  static_assert(MF_ME2_GG_TTGG_LANES_NEV == 31 && MF_ME2_GG_TTGG_LANES_EV_K == 15 && MF_LANES_EVT % 2 == 1, "generator input layout changed");
  const int lane = threadIdx.x & 31, lane4 = lane & 3;
  T* V = tile + MF_ME2_GG_TTGG_LANES_SLOTS * 32;
  T* E = V + MF_ME2_GG_TTGG_LANES_NV * 32 + (lane >> 2) * MF_LANES_EVT;
  T* Gp = E + MF_ME2_GG_TTGG_LANES_NEV;
  {                                                     // lane l publishes global gluon l; lanes 0, 1, 2 the quark line's inputs
    const T E0 = T(0.5) * rts, r2 = T(1.41421356237309504880);
    T kg[4], pf[4], o[5], f[5];
#pragma unroll
    for (int c = 0; c < 4; ++c) { kg[c] = (lane4 == 3) ? k[3][c] : k[2][c]; pf[c] = (lane4 == 2) ? k[1][c] : k[0][c]; }
    mf_gluon_ing<T>(kg, o);                             // eps / sqrt2 of an outgoing gluon
    mf_fermion_ing<T>(pf, T(P.m_top), f);
    const bool inc = lane4 < 2;
    const T sg = (lane4 == 0) ? T(1.0) : T(-1.0);
    T* Kt = E + MF_ME2_GG_TTGG_LANES_EV_K + lane4 * 4;
    Kt[0] = inc ? E0 : -kg[0]; Kt[1] = inc ? T(0.0) : -kg[1]; Kt[2] = inc ? T(0.0) : -kg[2]; Kt[3] = inc ? sg * E0 : -kg[3];
    T* Gl = Gp + lane4 * 6;
    Gl[0] = inc ? T(1.0) : r2 * o[0]; Gl[1] = inc ? T(0.0) : r2 * o[1]; Gl[2] = inc ? T(0.0) : r2 * o[2];
    Gl[3] = inc ? T(0.0) : r2 * o[3]; Gl[4] = inc ? sg : r2 * o[4]; Gl[5] = T(0.0);
    if (lane4 == 0) {
      E[MF_ME2_GG_TTGG_LANES_EV_MT] = T(P.m_top);
#pragma unroll
      for (int c = 0; c < 4; ++c) E[MF_ME2_GG_TTGG_LANES_EV_P4E + c] = k[1][c];
    } else if (lane4 < 3) {
      T* F = E + (lane4 == 1 ? MF_ME2_GG_TTGG_LANES_EV_T_WP : MF_ME2_GG_TTGG_LANES_EV_B_WP);
#pragma unroll
      for (int c = 0; c < 5; ++c) F[c] = f[c];
    }
  }
  __syncwarp();
  const int b4 = lane & ~3;
  T acc = mf_me2_gg_ttgg_lanes<T>(E, Gp, tile, V, lane4, lane, b4 | ((lane4 + 1) & 3), b4 | ((lane4 + 2) & 3), b4 | ((lane4 + 3) & 3));
  acc += __shfl_xor_sync(0xffffffffu, acc, 1);
  acc += __shfl_xor_sync(0xffffffffu, acc, 2);
  return T(P.me_pref) * acc;
}

// the same for a warp whose 32 lanes hold one event each: four rounds of eight events
template <typename T>
__device__ __forceinline__ T mf_me2_ttgg_warp32(const MfParams& P, T rts, const T k[4][4], T* tile) {
  const int lane = threadIdx.x & 31;
  T out = T(0.0);
#pragma unroll 1
  for (int r = 0; r < 4; ++r) {
    const int src = r * 8 + (lane >> 2);
    T kr[4][4];
#pragma unroll
    for (int p = 0; p < 4; ++p)
#pragma unroll
      for (int c = 0; c < 4; ++c) kr[p][c] = __shfl_sync(0xffffffffu, k[p][c], src);
    const T rr = __shfl_sync(0xffffffffu, rts, src);
    const T m = mf_me2_ttgg_group<T>(P, rr, kr, tile);
    const T t = __shfl_sync(0xffffffffu, m, 4 * (lane & 7));
    if ((lane >> 3) == r) out = t;
  }
  return out;
}
#endif

// ---- q q~ -> t t~ g (PROC 6) and q g -> t t~ q (PROC 7): the generated code takes generic external lines, so the other
// channels are the same code on relabelled momenta.  ch bit 0: the beams exchanged (the light quark comes along -z);
// bit 1: the charge-conjugate channel = t and t~ exchanged (q~ g -> t t~ q~).  DESIGN.md 5.10.
template <int PROC, typename T>
MF_HD T mf_me2_2q(const MfParams& P, T rts, const T k[3][4], int ch) {
  static_assert(MF_ME2_QQ_TTG_NIN == 41 && MF_ME2_QG_TTQ_NIN == 41, "generator input layout changed");
  T in[41];
  const T E = T(0.5) * rts, sz = (ch & 1) ? T(-1.0) : T(1.0), r2 = T(1.41421356237309504880);
  const T pa[4] = {E, T(0.0), T(0.0), sz * E}, pb[4] = {E, T(0.0), T(0.0), -sz * E};
  T k1[4], k2[4], f[5], o[5];
#pragma unroll
  for (int c = 0; c < 4; ++c) { k1[c] = (ch & 2) ? k[1][c] : k[0][c]; k2[c] = (ch & 2) ? k[0][c] : k[1][c]; }
  in[0] = T(P.m_top);
#pragma unroll
  for (int c = 0; c < 4; ++c) in[1 + c] = k2[c];
  mf_fermion_ing<T>(k1, T(P.m_top), in + 5);
  mf_fermion_ing<T>(k2, T(P.m_top), in + 10);
#pragma unroll
  for (int c = 0; c < 4; ++c) {                          // light line: u(pa) ... vbar(pb) (PROC 6) or ubar(k3) (PROC 7); gluon all-incoming
    in[15 + c] = pa[c];
    in[19 + c] = PROC == 6 ? pb[c] : -k[2][c];
    in[31 + c] = PROC == 6 ? -k[2][c] : pb[c];
  }
  mf_fermion_ing<T>(pa, T(0.0), f);
  in[23] = f[0]; in[24] = f[2]; in[25] = f[3]; in[26] = f[4];
  mf_fermion_ing<T>(PROC == 6 ? pb : k[2], T(0.0), f);
  in[27] = f[0]; in[28] = f[2]; in[29] = f[3]; in[30] = f[4];
  mf_gluon_ing<T>(PROC == 6 ? k[2] : pb, o);              // eps1, eps2 / sqrt2 of the gluon (linear basis: same vectors in and out)
  in[35] = r2 * o[0]; in[36] = r2 * o[1]; in[37] = r2 * o[2]; in[38] = r2 * o[3]; in[39] = r2 * o[4]; in[40] = T(0.0);
  return T(P.me_pref) * (PROC == 6 ? mf_me2_qq_ttg<T>(in) : mf_me2_qg_ttq<T>(in));
}

// S7 weighted with the parton luminosities: process 5 returns xg(x1) xg(x2) |M_gg|^2 + (L12 + L21) |M_qq|^2 (lum = the two
// luminosities from the front end); every other process its |M|^2
template <int PROC, typename T>
MF_HD T mf_me2_lum(const MfParams& P, T rts, const T k[MfProc<PROC>::N][4], const double* lum) {
  if constexpr (PROC == 5) return T(lum[0]) * mf_me2<1, T>(P, rts, k) + T(lum[1]) * mf_me2<4, T>(P, rts, k);
  else if constexpr (PROC == 6 || PROC == 7) {           // sum over the channels: one copy of the |M|^2 code
    T sum = T(0.0);
#if defined(__CUDACC__)
#pragma unroll 1
#endif
    for (int ch = 0; ch < MfChannels<PROC>::value; ++ch) sum += T(lum[ch]) * mf_me2_2q<PROC, T>(P, rts, k, ch);
    return sum;
  } else return mf_me2<PROC == 3 ? 1 : PROC, T>(P, rts, k);      // (process 3: mf_me2_ttgg_group instead)
}

// Front end of one event, S1-S6 + the weight prefactor: F = pref * |M|^2 for a passing event with
//   config 0   : pref = J_V (1/(8 pi)) K / (2 s)
//   configs 1-3: pref = J_V J_x f_g(x1) f_g(x2) S_f W_0 W_m K / (2 shat)
// edges: [d][nb+1], pdf_tab: [nx][nq] (both in shared memory on the device).  Returns the cut flag.
template <int PROC, bool REC, int CL = 0>
MF_HD bool mf_event_front(const MfParams& P, const double* edges, const double* pdf_tab, uint32_t iteration,
                          uint64_t ev, int bin[MfDim<PROC, CL>::D], double k[MfProc<PROC>::N][4], double& rts,
                          double& pref, MfEventRec* rec, unsigned* okeys = nullptr, double* lum = nullptr) {
  constexpr int D = MfDim<PROC, CL>::D, N = MfProc<PROC>::N, NGL = MfProc<PROC>::NGL;
  static_assert(PROC != 0 || CL == 0, "generator variants apply to processes 1-3");
  double u[D], y[D];
  mf_uniforms<D>(P, iteration, ev, u);                                   // S1
  const double JV = mf_vegas_map<D>(edges, P.nb, u, y, bin);             // S2
  double x1 = 1.0, x2 = 1.0, shat = P.s, jx = 1.0, lx1 = 0.0, lx2 = 0.0;
  if (PROC != 0) {                                                       // S3 / S3'
    if (CL != 0 && (P.gen & MFD_GEN_LINEAR)) mf_x_map_linear(P, y[0], y[1], x1, x2, shat, jx, lx1, lx2);
    else mf_x_map(P, y[0], y[1], x1, x2, shat, jx, lx1, lx2);
  }
  const double wps = CL == 1 ? mf_phase_space_classic<N>(shat, P.m_top, y + 2, k)                            // S4'
                        : mf_phase_space<N>(shat, PROC == 0 ? 0.0 : P.m_top, y + (PROC == 0 ? 0 : 2), k);   // S4
  rts = sqrt(shat);
  const bool pass = mf_cuts<NGL>(P, (const double(*)[4])(&k[0][0] + 8), x1, x2);   // S5 (final gluons = k[2..])
  double ff = 1.0, xf1 = 0.0, xf2 = 0.0;                                 // ff = f_g(x1) f_g(x2) / shat
  if (PROC == 7) {                                                       // S6q: q g, g q, q~ g, g q~ luminosities (to S7: mf_me2_lum)
    ff = 1.0 / (x1 * x2 * shat);
    if (REC || pass) {
      const double g1 = mf_pdf_strided<MF_NFL>(P, pdf_tab + 5, lx1, P.pdf_lq), g2 = mf_pdf_strided<MF_NFL>(P, pdf_tab + 5, lx2, P.pdf_lq);
      double q1 = 0.0, a1 = 0.0, q2 = 0.0, a2 = 0.0;
#pragma unroll
      for (int q = 1; q <= 5; ++q) {
        q1 += mf_pdf_strided<MF_NFL>(P, pdf_tab + 5 + q, lx1, P.pdf_lq); a1 += mf_pdf_strided<MF_NFL>(P, pdf_tab + 5 - q, lx1, P.pdf_lq);
        q2 += mf_pdf_strided<MF_NFL>(P, pdf_tab + 5 + q, lx2, P.pdf_lq); a2 += mf_pdf_strided<MF_NFL>(P, pdf_tab + 5 - q, lx2, P.pdf_lq);
      }
      lum[0] = q1 * g2; lum[1] = g1 * q2; lum[2] = a1 * g2; lum[3] = g1 * a2;
      xf1 = lum[0] + lum[2]; xf2 = lum[1] + lum[3];                      // the record: quark from beam 1 / from beam 2
    }
  } else if (PROC == 6) {                                                // q q~ and q~ q luminosities (the two |M|^2 differ)
    ff = 1.0 / (x1 * x2 * shat);
    if (REC || pass) { mf_lumi_qq(P, pdf_tab, lx1, lx2, P.pdf_lq, xf1, xf2); lum[0] = xf1; lum[1] = xf2; }
  } else if (MfPdf<PROC>::FLAVOURS) {                                    // S6q: flavour-summed luminosity (xf1, xf2 = the two sums)
    mf_lumi_qq(P, pdf_tab, lx1, lx2, P.pdf_lq, xf1, xf2);
    ff = (xf1 + xf2) / (x1 * x2 * shat);
    if (PROC == 5) {                                                     // both subprocesses: the luminosities go to S7 (mf_me2_lum)
      const double g1 = mf_pdf_strided<MF_NFL>(P, pdf_tab + 5, lx1, P.pdf_lq), g2 = mf_pdf_strided<MF_NFL>(P, pdf_tab + 5, lx2, P.pdf_lq);
      lum[0] = g1 * g2; lum[1] = xf1 + xf2;
      xf1 = lum[0]; xf2 = lum[1];                                        // the record holds the two luminosities
      ff = 1.0 / (x1 * x2 * shat);
    }
  } else if (PROC != 0 && (REC || pass)) {                               // S6
    xf1 = mf_pdf(P, pdf_tab, lx1, P.pdf_lq);
    xf2 = mf_pdf(P, pdf_tab, lx2, P.pdf_lq);
    ff = xf1 * xf2 / (x1 * x2 * shat);                                   // f_g = xf / x: one division for the three
  } else {
    ff = 1.0 / shat;
  }
  pref = JV * jx * ff * wps * P.wconst;                                  // S8 without |M|^2
  if (okeys) *okeys = (P.n_obs > 0 && pass) ? mf_obs_keys<N>(P, (const double(*)[4])k) : 0u;
  if (REC) {
#pragma unroll
    for (int j = 0; j < D; ++j) rec->y[j] = y[j];
    const double E = 0.5 * rts;
    rec->mom[0][0] = E; rec->mom[0][1] = 0.0; rec->mom[0][2] = 0.0; rec->mom[0][3] = E;
    rec->mom[1][0] = E; rec->mom[1][1] = 0.0; rec->mom[1][2] = 0.0; rec->mom[1][3] = -E;
#pragma unroll
    for (int i = 0; i < N; ++i)
#pragma unroll
      for (int c = 0; c < 4; ++c) rec->mom[2 + i][c] = k[i][c];
    rec->pdf[0] = xf1; rec->pdf[1] = xf2; rec->pass = pass ? 1 : 0;
  }
  return pass;
}

// One whole event: front end, then S7 and S8.  bin[] receives the VEGAS bins; rec (nullable) the
// debug record.
template <int PROC, bool REC, typename T = double, int CL = 0>
MF_HD double mf_event(const MfParams& P, const double* edges, const double* pdf_tab,
                      uint32_t iteration, uint64_t ev, int bin[MfDim<PROC, CL>::D], bool& pass,
                      MfEventRec* rec, unsigned* okeys = nullptr) {
  constexpr int N = MfProc<PROC>::N;
  double k[N][4], rts, pref, lum[MF_NLUM] = {0.0, 0.0, 0.0, 0.0};
  pass = mf_event_front<PROC, REC, CL>(P, edges, pdf_tab, iteration, ev, bin, k, rts, pref, rec, okeys, lum);
  double me2 = 0.0;
  if (MF_UNIFORM_ME || pass) {                                           // S7 (in the real type T)
    T kt[N][4];
#pragma unroll
    for (int i = 0; i < N; ++i)
#pragma unroll
      for (int c = 0; c < 4; ++c) kt[i][c] = (T)k[i][c];
    me2 = (double)mf_me2_lum<PROC, T>(P, (T)rts, kt, lum);
  }
  if (!pass) me2 = 0.0;
  if (REC) rec->me2 = MfChannels<PROC>::value > 1 ? me2 / (lum[0] + lum[1] + lum[2] + lum[3]) : me2;   // several channels: the luminosity-weighted mean |M|^2
  return pass ? pref * me2 : 0.0;                                        // S8
}
