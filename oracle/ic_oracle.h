/*
 * oracle/ic_oracle.h -- interface of the CPU oracle.  TEST INFRASTRUCTURE ONLY
 * (see the header of ic_oracle.c).  Nothing under paper_2301_11735_b200/ may
 * include this file.
 */
#ifndef IC_ORACLE_H
#define IC_ORACLE_H
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* State of one lattice copy besides the site codes themselves (the codes live
 * in a caller-owned int8 array of Lx*Ly entries, row-major, code[y*Lx+x]).    */
typedef struct {
  int32_t Lx, Ly;
  int32_t replica;          /* counter field of the random-number address       */
  int32_t pad_;
  double delta, V, J;       /* parameters of eq. (1)/(3)                        */
  uint64_t seed;            /* Philox key                                       */
  uint64_t sweep;           /* global sweep counter since creation              */
  int64_t n2, bV, bJ, M, Ms, Q; /* exact integers, tracked incrementally        */
  int64_t nmeas;
  double sumE, sumE2, sumM, sumM2, sumAbsM, sumMs, sumMs2, sumAbsMs;
  int64_t n_attempt, n_accept, n_null; /* statistics                            */
} orc_state;

#ifndef ORC_UPDATE_ROUNDS
#define ORC_UPDATE_ROUNDS 7 /* Philox rounds of the update stream (G5); the default of orc_set_update_rounds */
#endif
int orc_set_update_rounds(int rounds); /* 1..16; 0 on success.  Not to be called while a sweep runs. */
int orc_get_update_rounds(void);
void orc_philox4x32(const uint32_t ctr[4], const uint32_t key[2], int rounds, uint32_t out[4]);
void orc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]);
void orc_philox_tagged(uint64_t seed, uint32_t c0, uint32_t c1, uint32_t c2, uint32_t replica, uint32_t tag, uint32_t out[4]);

uint32_t orc_threshold(double delta, double V, double J, int dn2, int dV, int dJ, double T);
void orc_recompute(const int8_t* code, int Lx, int Ly, int64_t out6[6]);
int orc_pair_table(int q, int idx, int8_t out2[2]);
int orc_pair_update(orc_state* st, int8_t* code, int xa, int ya, int xb, int yb, uint32_t w, double T);
void orc_init_state(int8_t* code, int Lx, int Ly, int64_t nplus, int64_t nminus, uint64_t seed, int replica);
void orc_attach(orc_state* st, const int8_t* code);
void orc_reset_observables(orc_state* st);
void orc_schedule_params(int L, uint64_t seed, uint64_t sweep, int32_t out4[4]);
int64_t orc_schedule_s1(int L, uint64_t seed, uint64_t sweep, int phase, int64_t* ia, int64_t* ib,
                        uint32_t* c0, uint32_t* c1, uint32_t* word);
int orc_sweep_s1(orc_state* st, int8_t* code, double T, int64_t nsweeps, int order, int64_t* trace);
int orc_sweep_s1_mt(orc_state* st, int8_t* code, double T, int64_t nsweeps, int nthreads, int64_t* trace);
int orc_sweep_s0(orc_state* st, int8_t* code, double T, int64_t nsweeps, int64_t* trace);
void orc_measure(orc_state* st, int64_t* trace_row);

/* ic_variants.c: what the paper describes around the main algorithm (negative controls, maps, drop observable) */
int orc_sweep_nn(orc_state* st, int8_t* code, double T, int64_t nsweeps, int64_t* trace);
int orc_sweep_mu(orc_state* st, int8_t* code, double T, int64_t nsweeps, double* mu, double kappa, int64_t q_target,
                 int64_t* trace);
int64_t orc_build_map_paper(int Lx, int Ly, uint64_t seed, uint64_t map_index, int64_t npairs, int64_t* ia, int64_t* ib);
int64_t orc_build_map_luby(int Lx, int Ly, uint64_t seed, uint64_t map_index, int64_t K, int64_t* ia, int64_t* ib, uint8_t* alive);
int orc_sweep_maps(orc_state* st, int8_t* code, double T, int64_t nmaps, int mode, int64_t K, int64_t* trace, int64_t* attempted);
int orc_largest_cluster(const int8_t* code, int Lx, int Ly, int which, int64_t out2[2]);

/* ic_enum.c: exact enumeration */
int64_t orc_enum_bruteforce(int Lx, int Ly, int64_t* keys /* [cap][6] */, uint64_t* counts, int64_t cap);
int64_t orc_enum_rows(int Lx, int Ly, int nthreads, int64_t* keys /* [cap][4] */, uint64_t* counts,
                      uint64_t* sumM2, uint64_t* sumMs2, int64_t cap);

#ifdef __cplusplus
}
#endif
#endif
