/* bz_testhooks.h -- test-only export of libbz_testhooks.so (NOT part of the product's C ABI, include/bz.h).
 *
 * The per-sample channel algebra (S8c steps 4-6: Table I; bracket of Eq. 5; deposits of Eq. 22,
 * P:201) run ON THE HOST through the same inline functions the kernels use, so that the factorised form can be checked
 * against the per-channel definition without a GPU.
 *   fv_host[slot*7 + id], slot 0..3 = cells i, j, k, l, id = species id (inactive ids ignored);
 *   out_host[slot*7 + id] = deposit in number units for weight w (= K/(E1 E2));
 *   variant 0 = deposit<> (the whole bracket), 1 = deposit_half<> twice (gain + loss halves, as collide_kernel does).
 * Returns 0, or -1 on a bad argument. */
#ifndef BZ_TESTHOOKS_H
#define BZ_TESTHOOKS_H
#ifdef __cplusplus
extern "C" {
#endif
int bz_debug_deposit_host(const int* species, int n_species, double alpha_s, const double* fv_host,
                          double s, double t, double u, double m2, double w, int variant, double* out_host);
#ifdef __cplusplus
}
#endif
#endif
