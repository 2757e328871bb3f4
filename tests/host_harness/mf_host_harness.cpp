// TEST HARNESS ONLY (never part of the product library): compiles the product's per-event device
// functions (csrc/mf_event.cuh, including the generated |M|^2 code) for the host with g++, so that
// the CPU test-suite can check that arithmetic event by event against the oracle without a GPU.
// gg -> tt~gg spreads one event over four lanes that exchange currents through a shared tile between warp barriers
// (gen/lanes.py): the harness runs the generated per-lane code on four host threads, __syncwarp() = a std::barrier.
#include <barrier>
#include <thread>
#include <cstring>
static std::barrier<> g_lane_barrier(4);
static inline void __syncwarp() { g_lane_barrier.arrive_and_wait(); }
#define MF_LANES_HOST_EMULATION
#include "../../paper_2105_10529_b200/csrc/mf_event.cuh"
#include "../../paper_2105_10529_b200/csrc/mf_params.h"

// host stand-in of mf_me2_ttgg_group (mf_event.cuh): same event table, same per-lane call
static double ttgg_lanes_host(const MfParams& P, double rts, const double k[4][4]) {
  constexpr int SL = MF_ME2_GG_TTGG_LANES_SLOTS, NV = MF_ME2_GG_TTGG_LANES_NV, NEV = MF_ME2_GG_TTGG_LANES_NEV;
  static double tile[(SL + NV) * 32 + NEV + 24];
  double* V = tile + SL * 32;
  double* E = V + NV * 32;
  double* Gp = E + NEV;
  const double E0 = 0.5 * rts, r2 = 1.41421356237309504880;
  E[MF_ME2_GG_TTGG_LANES_EV_MT] = P.m_top;
  for (int c = 0; c < 4; ++c) E[MF_ME2_GG_TTGG_LANES_EV_P4E + c] = k[1][c];
  mf_fermion_ing<double>(k[0], P.m_top, E + MF_ME2_GG_TTGG_LANES_EV_T_WP);
  mf_fermion_ing<double>(k[1], P.m_top, E + MF_ME2_GG_TTGG_LANES_EV_B_WP);
  for (int l = 0; l < 4; ++l) {
    const bool inc = l < 2;
    const double sg = l == 0 ? 1.0 : -1.0;
    const double* kg = l == 3 ? k[3] : k[2];
    double o[5];
    mf_gluon_ing<double>(kg, o);
    double* Kt = E + MF_ME2_GG_TTGG_LANES_EV_K + 4 * l;
    Kt[0] = inc ? E0 : -kg[0]; Kt[1] = inc ? 0.0 : -kg[1]; Kt[2] = inc ? 0.0 : -kg[2]; Kt[3] = inc ? sg * E0 : -kg[3];
    Gp[l * 6 + 0] = inc ? 1.0 : r2 * o[0]; Gp[l * 6 + 1] = inc ? 0.0 : r2 * o[1]; Gp[l * 6 + 2] = inc ? 0.0 : r2 * o[2];
    Gp[l * 6 + 3] = inc ? 0.0 : r2 * o[3]; Gp[l * 6 + 4] = inc ? sg : r2 * o[4]; Gp[l * 6 + 5] = 0.0;
  }
  double acc[4];
  std::thread th[4];
  for (int l = 0; l < 4; ++l) th[l] = std::thread([&, l] {
    acc[l] = mf_me2_gg_ttgg_lanes<double>(E, Gp, tile, V, l, l, (l + 1) & 3, (l + 2) & 3, (l + 3) & 3);
  });
  for (int l = 0; l < 4; ++l) th[l].join();
  return P.me_pref * ((acc[0] + acc[1]) + (acc[2] + acc[3]));
}
template <int CL>
static double event_ttgg(const MfParams& P, const double* edges, const double* pdf, uint32_t it, uint64_t ev, int* bin, bool& ok, MfEventRec* rec) {
  double k[4][4], rts, pref;
  ok = mf_event_front<3, true, CL>(P, edges, pdf, it, ev, bin, k, rts, pref, rec);
  rec->me2 = ok ? ttgg_lanes_host(P, rts, k) : 0.0;
  return ok ? pref * rec->me2 : 0.0;
}

template <int PROC>
static double run(const MfParams& P, const double* edges, const double* pdf, uint32_t it, uint64_t ev,
                  int* bins, int* pass, double* rec_out) {
  int bin[MfProc<PROC>::D]; bool ok; MfEventRec rec;
  std::memset(&rec, 0, sizeof rec);
  double F;
  if constexpr (PROC == 3) F = event_ttgg<0>(P, edges, pdf, it, ev, bin, ok, &rec);
  else F = mf_event<PROC, true>(P, edges, pdf, it, ev, bin, ok, &rec);
  for (int j = 0; j < MfProc<PROC>::D; ++j) bins[j] = bin[j];
  *pass = ok;
  // rec_out: y[10], mom[24], me2, pdf[2]
  std::memcpy(rec_out, rec.y, sizeof(double) * 10);
  std::memcpy(rec_out + 10, rec.mom, sizeof(double) * 24);
  rec_out[34] = rec.me2; rec_out[35] = rec.pdf[0]; rec_out[36] = rec.pdf[1];
  return F;
}

extern "C" double mfh_event(const MfParams* P, const double* edges, const double* pdf, uint32_t it,
                            uint64_t ev, int* bins, int* pass, double* rec_out) {
  switch (P->process) {
    case 0: return run<0>(*P, edges, pdf, it, ev, bins, pass, rec_out);
    case 1: return run<1>(*P, edges, pdf, it, ev, bins, pass, rec_out);
    case 2: return run<2>(*P, edges, pdf, it, ev, bins, pass, rec_out);
    case 4: return run<4>(*P, edges, pdf, it, ev, bins, pass, rec_out);   // pdf: the library's flavour slice (mfh_flavour_slice)
    case 5: return run<5>(*P, edges, pdf, it, ev, bins, pass, rec_out);
    case 6: return run<6>(*P, edges, pdf, it, ev, bins, pass, rec_out);
    case 7: return run<7>(*P, edges, pdf, it, ev, bins, pass, rec_out);
#ifndef MFH_NO_TTGG
    case 3: return run<3>(*P, edges, pdf, it, ev, bins, pass, rec_out);
#endif
  }
  return -1.0;
}
// gg -> tt~g with the |M|^2 stage in fp32 (the product's precision = 32 variant), same record layout
extern "C" double mfh_event_ttg_f32(const MfParams* P, const double* edges, const double* pdf, uint32_t it,
                                    uint64_t ev, int* bins, int* pass, double* rec_out) {
  int bin[MfProc<2>::D]; bool ok; MfEventRec rec;
  std::memset(&rec, 0, sizeof rec);
  double F = mf_event<2, true, float>(*P, edges, pdf, it, ev, bin, ok, &rec);
  for (int j = 0; j < MfProc<2>::D; ++j) bins[j] = bin[j];
  *pass = ok;
  std::memcpy(rec_out, rec.y, sizeof(double) * 10);
  std::memcpy(rec_out + 10, rec.mom, sizeof(double) * 24);
  rec_out[34] = rec.me2; rec_out[35] = rec.pdf[0]; rec_out[36] = rec.pdf[1];
  return F;
}
// selectable generators: classic 4n-random RAMBO (P->gen & 1; d = 2 + 4 n_final) and/or the linear-tau
// map (P->gen & 2, run-time branch).  rec_out: y[18], mom[24], me2, pdf[2]
template <int PROC, int CL>
static double run_gen(const MfParams& P, const double* edges, const double* pdf, uint32_t it, uint64_t ev,
                      int* bins, int* pass, double* rec_out) {
  int bin[MfDim<PROC, CL>::D]; bool ok; MfEventRec rec;
  std::memset(&rec, 0, sizeof rec);
  double F;
  if constexpr (PROC == 3) F = event_ttgg<CL>(P, edges, pdf, it, ev, bin, ok, &rec);
  else F = mf_event<PROC, true, double, CL>(P, edges, pdf, it, ev, bin, ok, &rec);
  for (int j = 0; j < MfDim<PROC, CL>::D; ++j) bins[j] = bin[j];
  *pass = ok;
  std::memcpy(rec_out, rec.y, sizeof(double) * 18);
  std::memcpy(rec_out + 18, rec.mom, sizeof(double) * 24);
  rec_out[42] = rec.me2; rec_out[43] = rec.pdf[0]; rec_out[44] = rec.pdf[1];
  return F;
}
extern "C" double mfh_event_gen(const MfParams* P, const double* edges, const double* pdf, uint32_t it,
                                uint64_t ev, int* bins, int* pass, double* rec_out) {
  const bool cl = P->gen & MFD_GEN_CLASSIC;
  switch (P->process) {
    case 1: return cl ? run_gen<1, 1>(*P, edges, pdf, it, ev, bins, pass, rec_out) : run_gen<1, 2>(*P, edges, pdf, it, ev, bins, pass, rec_out);
    case 5: return cl ? run_gen<5, 1>(*P, edges, pdf, it, ev, bins, pass, rec_out) : run_gen<5, 2>(*P, edges, pdf, it, ev, bins, pass, rec_out);
    case 4: return cl ? run_gen<4, 1>(*P, edges, pdf, it, ev, bins, pass, rec_out) : run_gen<4, 2>(*P, edges, pdf, it, ev, bins, pass, rec_out);
    case 2: return cl ? run_gen<2, 1>(*P, edges, pdf, it, ev, bins, pass, rec_out) : run_gen<2, 2>(*P, edges, pdf, it, ev, bins, pass, rec_out);
    case 6: return cl ? run_gen<6, 1>(*P, edges, pdf, it, ev, bins, pass, rec_out) : run_gen<6, 2>(*P, edges, pdf, it, ev, bins, pass, rec_out);
    case 7: return cl ? run_gen<7, 1>(*P, edges, pdf, it, ev, bins, pass, rec_out) : run_gen<7, 2>(*P, edges, pdf, it, ev, bins, pass, rec_out);
#ifndef MFH_NO_TTGG
    case 3: return cl ? run_gen<3, 1>(*P, edges, pdf, it, ev, bins, pass, rec_out) : run_gen<3, 2>(*P, edges, pdf, it, ev, bins, pass, rec_out);
#endif
  }
  return -1.0;
}
// the library's device copy of the 11-flavour grid (mf_params.h mf_flavour_slice); returns its length in doubles
extern "C" int mfh_flavour_slice(const MfParams* P, const double* pdf11, double* out) {
  if (out) mf_flavour_slice(*P, pdf11, out);
  return P->pdf_smem;
}
extern "C" int mfh_params_size(void) { return (int)sizeof(MfParams); }
extern "C" int mfh_fill_params(const mf_config_t* c, MfParams* P) { std::string e; return mf_fill_params(c, P, e); }
