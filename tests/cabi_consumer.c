/* A plain C99 consumer of include/gf.h: proves that the header compiles as C and that libgf.so links from C.  It only
 * walks error paths that return before any device work (no GPU needed). */
#include <stdio.h>
#include <string.h>

#include "gf.h"

#define CHECK(cond)                                            \
  do {                                                         \
    if (!(cond)) {                                             \
      fprintf(stderr, "cabi_consumer: failed: %s\n", #cond);   \
      return 1;                                                \
    }                                                          \
  } while (0)

int main(void) {
  gf_ctx* ctx = (gf_ctx*)0x1;
  double F = 0.0, theta = 0.0, tflops = 0.0;
  int done = -1;
  size_t bytes;

  bytes = gf_workspace_bytes(8, 8, 8, 8, GF_FP64, 18);
  CHECK(bytes >= (size_t)4 * 4096 * 144);
  CHECK(gf_workspace_bytes(7, 8, 8, 8, GF_FP64, 18) == 0); /* odd extent */
  CHECK(gf_workspace_bytes(8, 8, 8, 8, GF_FP32, 10) == 0); /* storage must be 18, 12 or 8 */
  CHECK(gf_workspace_bytes_sun(5, 8, 8, 8, 8, GF_FP64) == 0 && gf_workspace_bytes_sun(4, 8, 8, 8, 8, GF_FP64) > 0);

  CHECK(gf_create(NULL, 8, 8, 8, 8, GF_LANDAU, GF_FP64, 18, NULL, 0, NULL) == GF_EINVAL);
  CHECK(gf_create(&ctx, 8, 8, 8, 9, GF_LANDAU, GF_FP64, 18, NULL, 0, NULL) == GF_EODD && ctx == NULL);
  CHECK(gf_create(&ctx, 8, 8, 8, 8, 7, GF_FP64, 18, NULL, 0, NULL) == GF_EUNSUPPORTED);
  CHECK(gf_create(&ctx, 8, 8, 8, 8, GF_COULOMB, GF_FP64, 10, NULL, 0, NULL) == GF_EUNSUPPORTED);
  CHECK(gf_create(&ctx, 8, 8, 8, 8, GF_COULOMB, GF_FP64, 12, NULL, 0, NULL) == GF_EINVAL); /* null workspace */

  CHECK(gf_set_links(NULL, NULL) == GF_EINVAL);
  CHECK(gf_ovr_sweep(NULL, 1, 1.7) == GF_EINVAL);
  CHECK(gf_measure(NULL, &F, &theta) == GF_EINVAL);
  CHECK(gf_fix(NULL, 1.7, 1e-12, 10, 1, &done) == GF_EINVAL);
  CHECK(gf_reunitarize(NULL) == GF_EINVAL);
  CHECK(gf_peak_fma(GF_FP64, 0.0, NULL, NULL, &tflops) == GF_EINVAL);
  CHECK(gf_fix_plan(1.7, 1e-12, 100, 10, 95, 1.0, &done) == GF_OK && done == 5);
  CHECK(gf_fix_plan(1.7, 1e-12, 100, 10, 40, 1e-13, &done) == GF_OK && done == 0);
  CHECK(gf_fix_plan(2.0, 1e-12, 100, 10, 0, 1.0, &done) == GF_EINVAL);
  {
    const double Fs[2] = {0.25, 0.75}, ts[2] = {2.0, 4.0};
    CHECK(gf_combine_slabs(Fs, ts, 2, &F, &theta) == GF_OK && F == 0.5 && theta == 3.0);
  }
  CHECK(gf_kernel_launches(NULL) == 0);
  CHECK(strcmp(gf_strerror(GF_OK), "ok") == 0);
  CHECK(strlen(gf_strerror(GF_EODD)) > 0 && strlen(gf_last_error(NULL)) == 0);
  gf_destroy(NULL);
  puts("cabi_consumer: ok");
  return 0;
}
