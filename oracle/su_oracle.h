/*
 * su_oracle.h — C interface of the CPU ORACLE for the SU(Nc) heatbath + overrelaxation sweep
 * of Cardoso & Bicudo, arXiv:1112.4533.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT. Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may load it. It shares no code, header,
 * table or constant generator with the CUDA path under paper_1112_4533_b200/csrc.
 *
 * It is a plain, slow, step-by-step restatement of the method: complex Nc x Nc matrices in
 * std::complex<T> (T = float or double, the lattice precision; "precision by
 * templates"), lexicographic site loops, the paper's order of operations:
 *   staple (eq 9) -> W = U S^dagger (step 2)
 *   -> for every SU(2) subgroup (i<j) (steps 3-5): project (eq 11), heatbath
 *      draw (eqs 12-14) or overrelaxation (eq 17), left-multiply (eq 15).
 * Readings of ambiguous passages are the R1..R19 of DESIGN.md.
 *
 * Parity pins: see tests/test_oracle_*.py. Unpinned beyond invariants + GPU agreement:
 *   thermalised means of SU(4) beta=11.0 and SU(6) beta=25.0 ("parity unpinned" for those
 *   two numbers only; every function below has at least one pin that is not itself).
 *
 * All functions return 0 on success, non-zero on invalid arguments. No exceptions cross.
 */
#ifndef SU_ORACLE_H
#define SU_ORACLE_H
#include <stddef.h>
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

typedef struct so_lattice so_lattice;

/* precision: 0 = float, 1 = double.  recon12: 1 = SU(3) two-row storage emulation
 * (third row rebuilt as conj(row0 x row1) whenever a link is stored). */
int  so_create(int Nc, int Lx, int Ly, int Lz, int Lt, int precision, int recon12, so_lattice** out);
void so_destroy(so_lattice*);

int so_init_cold(so_lattice*, uint64_t seed);               /* PAPER.md:164 cold start */
int so_init_hot (so_lattice*, uint64_t seed);               /* PAPER.md:164 hot start (Haar) */
int so_set_rng  (so_lattice*, uint64_t seed, uint32_t sweep_counter);

/* One sweep = n_hb heatbath passes then n_or overrelaxation passes; each pass = parity 0,1 x
 * mu 0..3. Uses then increments the sweep counter. */
int so_sweep  (so_lattice*, double beta, int n_hb, int n_or);
/* One (parity, mu) sub-step. kind 0 = heatbath, 1 = overrelaxation. pass = heatbath pass number
 * (enters the RNG counter). attempts: NULL or n_sub * V/2 bytes, [subgroup][cb] with cb the
 * checkerboard index (lexicographic index / 2): KP attempts used (0 for OR / unchanged). */
int so_substep(so_lattice*, double beta, int kind, int pass, int parity, int mu, uint8_t* attempts);

int so_plaquette (so_lattice*, double* out);                /* eq 4; mean ReTr P / Nc */
int so_polyakov  (so_lattice*, double out[2]);              /* mean Tr prod_t U_3 / Nc */
int so_reunitarize(so_lattice*);

/* canonical layout [t][z][y][x][mu][row][col][re,im], doubles; n = 4V * 2Nc^2 */
int so_export_links(so_lattice*, double* dst, size_t n);
int so_import_links(so_lattice*, const double* src, size_t n);
int so_get_counters(so_lattice*, uint64_t* kp_attempts_total, uint64_t* kp_exhausted);

/* ---- hooks that expose single steps so the tests can pin them ---- */
void so_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]);
/* uniform in (0,1] from a 32-bit word, precision 0/1 (returned as double, exact) */
double so_uniform(uint32_t w, int precision);
/* staple S (eq 9 as printed) of link (site, mu), row-major re,im doubles (2 Nc^2) */
int so_staple(so_lattice*, size_t site, int mu, double* out);
/* n Kennedy-Pendleton draws at fixed alpha: sample i uses Philox counter c0 = i, c1 = 0,
 * c2 = kind<<28 (kind 0 attempts, 1 direction). out_v: 4n doubles (a0,a1,a2,a3);
 * out_attempts: n bytes (0 = exhausted). */
int so_kp_sample(int precision, double alpha, uint64_t seed, size_t n, double* out_v, uint8_t* out_attempts);
/* Apply the subgroup loop to ONE matrix pair outside any lattice (for maximisation pins):
 * U, W: Nc x Nc row-major re,im doubles, updated in place; kind 0/1; rng counter fields given. */
int so_update_matrix(int Nc, int precision, double beta, int kind, uint64_t seed,
                     uint32_t c0, uint32_t c1, uint32_t c2_base, double* U, double* W,
                     uint8_t* attempts /* n_sub */);
int so_num_threads(void);

#ifdef __cplusplus
}
#endif
#endif
