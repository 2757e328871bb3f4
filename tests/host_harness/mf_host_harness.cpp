// TEST HARNESS ONLY (never part of the product library): compiles the product's per-event device
// functions (csrc/mf_event.cuh, including the generated |M|^2 code) for the host with g++, so that
// the CPU test-suite can check that arithmetic event by event against the oracle without a GPU.
#include "../../paper_2105_10529_b200/csrc/mf_event.cuh"
#include "../../paper_2105_10529_b200/csrc/mf_params.h"
#include <cstring>

template <int PROC>
static double run(const MfParams& P, const double* edges, const double* pdf, uint32_t it, uint64_t ev,
                  int* bins, int* pass, double* rec_out) {
  int bin[MfProc<PROC>::D]; bool ok; MfEventRec rec;
  std::memset(&rec, 0, sizeof rec);
  double F = mf_event<PROC, true>(P, edges, pdf, it, ev, bin, ok, &rec);
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
  double F = mf_event<PROC, true, double, CL>(P, edges, pdf, it, ev, bin, ok, &rec);
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
