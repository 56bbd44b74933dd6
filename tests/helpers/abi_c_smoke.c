/* The boundary used from plain C, without Python or torch (include/mcdc.h): BASELINE.json config 1
 * (infinite medium, Sigma_t 1, Sigma_s 0.5; closed form: flux 1/Sigma_a = 2 per source particle,
 * PAPER-independent textbook value), workspace from cudaMalloc, results read into host memory.
 * Built and run by tests/test_gpu_parity.py::test_c_abi_from_plain_c. */
#include <math.h>
#include <stdio.h>
#include <stdint.h>
#include <cuda_runtime_api.h>
#include "mcdc.h"

int main(void)
{
  const double inf = INFINITY;
  double sigma_t[1] = {1.0}, sigma_c[1] = {0.5}, sigma_f[1] = {0.0}, nu[1] = {0.0}, sigma_s[1] = {0.5},
         chi[1] = {1.0}, speed[1] = {1.0};
  mcdc_materials mat = {1, 1, sigma_t, sigma_c, sigma_f, nu, sigma_s, chi, speed};
  double planes[2] = {-inf, inf}, radius[1] = {0.0};
  int32_t mo[1] = {0}, mi[1] = {-1};
  mcdc_geometry geo = {1, 1, 1, planes, planes, planes, mo, mi, radius, {0, 0, 0, 0, 0, 0}};
  double pdf[1] = {1.0};
  mcdc_source src = {0, {0, 0, 0}, {0, 0, 0}, 1, {1, 0, 0}, pdf, 0.0};
  double ts[2] = {0.0, inf};
  mcdc_tally_mesh tal = {1, 1, 1, 1, planes, planes, planes, ts, 0};
  mcdc_census cen = {0, NULL, 0};
  mcdc_problem *p = NULL;
  if (mcdc_problem_create(&mat, &geo, &src, &tal, &cen, &p) != MCDC_OK) { printf("create: %s\n", mcdc_last_error()); return 1; }
  mcdc_run_params rp = {0, 100000, 2, 0.0};
  size_t bytes = mcdc_workspace_bytes(p, &rp);
  void *ws = NULL;
  if (bytes == 0 || cudaMalloc(&ws, bytes) != cudaSuccess) { printf("workspace\n"); return 1; }
  if (mcdc_run(p, &rp, ws, bytes, NULL) != MCDC_OK) { printf("run: %s\n", mcdc_last_error()); return 1; }
  double flux = 0.0, se = 0.0;
  mcdc_counters c;
  if (mcdc_tally_size(p) != 1 || mcdc_tally_read(p, 0, &flux, 1, 0) != MCDC_OK || mcdc_tally_read(p, 1, &se, 1, 0) != MCDC_OK ||
      mcdc_counters_read(p, 0, -1, &c) != MCDC_OK) { printf("read: %s\n", mcdc_last_error()); return 1; }
  /* error paths: a NULL problem and a too small workspace are statuses, not crashes */
  if (mcdc_run(p, &rp, ws, 16, NULL) != MCDC_ENOMEM || mcdc_tally_read(NULL, 0, &flux, 1, 0) != MCDC_EINVAL) { printf("error paths\n"); return 1; }
  printf("flux %.6f se %.6f captures %llu collisions %llu\n", flux, se, (unsigned long long)c.captures, (unsigned long long)c.collisions);
  int ok = fabs(flux - 2.0) < 0.03 && se > 0.0 && se < 0.02 && c.captures == 100000 && c.source == 100000 &&
           c.collisions == c.scatters + c.captures;
  mcdc_problem_destroy(p);
  cudaFree(ws);
  printf(ok ? "OK\n" : "FAILED\n");
  return ok ? 0 : 1;
}
