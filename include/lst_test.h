/* lst_test.h -- test hooks of liblst_b200.so.  NOT part of the product API (include/lst.h).
 * lst_host_eval / lst_host_ls_window run the CUDA path's __host__ __device__ selection arithmetic
 * (csrc/lst_math.cuh) on the CPU so that the "-m not gpu" tests can compare it with the oracle without
 * a GPU.  lst_test_get_hit_index reads back what step a0 left in a slot.  HOST pointers only.
 */
#ifndef LST_TEST_H
#define LST_TEST_H
#include "lst.h"

#ifdef __cplusplus
extern "C" {
#endif

/* n candidates of one level.  pts: n * npts * 3 floats (x, y, z per point), cats: n * npts module
 * categories, aux: level-specific doubles, 4 per candidate.
 *   LST_MD : npts 2 (lower, upper hit), cats[0] = module category;          f: kappa, sigma_kappa, dphi
 *   LST_LS : npts 2 (anchors), aux = {kappa_i, sigma_i, kappa_o, sigma_o};   f: kappa, sigma_kappa, dphi
 *   LST_T3 : npts 3;                                                        f: kappa3, sigma_kappa3, beta
 *   LST_T5 : npts 5, aux = {kappa3_a, sigma_a, kappa3_b, sigma_b};          f: R, chi2, eta
 * pass[i] = the fp64 decision, pre[i] (may be NULL) = the fp32 pre-filter's verdict (1 where the
 * level has none), f (may be NULL): n * 3 doubles.  LST_EINVAL on a bad level / null pointer. */
int lst_host_eval(const lst_config *cfg /* NULL = defaults */, int level, uint32_t n, const float *pts,
                  const uint8_t *cats, const double *aux, uint8_t *pass, uint8_t *pre, double *f);

/* The per-(inner MD, connected module) window of the LS enumeration (ls_row_window): row = n * {rt, z}
 * of the inner anchor, row_cat its category; box = n * {rt min, rt max, z min, z max} of the module's
 * MD anchors, box_cat the module's category.  live[i] = 0: no anchor in the box can pass L1;
 * w[i]: bound on |dphi| of a pair that can pass L2 (> pi: none). */
int lst_host_ls_window(const lst_config *cfg, uint32_t n, const float *row, const uint8_t *row_cat, const float *box,
                       const uint8_t *box_cat, uint8_t *live, float *w);

/* Read-only view of step a0 of the slot's last run (synchronises the slot's stream): det_off
 * (2 * n_modules + 1 words), hit_orig (n_hits words) and hit_xyzr (4 * n_hits floats) as the chain's
 * k_hist / k_scatter / k_rank wrote them; any of the three may be NULL.  *n_hits_out (may be NULL) =
 * hits of the event.  Used by tests/test_zz_no_alloc.py to compare lst_index_hits_static with the
 * regular path.  LST_ESTATE before the first run of the slot. */
int lst_test_get_hit_index(lst_ctx *ctx, uint32_t slot, uint32_t *det_off, uint32_t *hit_orig, float *hit_xyzr,
                           uint32_t *n_hits_out);

#ifdef __cplusplus
}
#endif
#endif
