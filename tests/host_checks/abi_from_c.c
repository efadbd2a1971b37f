/* The C ABI from plain C99 (no C++, no Python): include/smcx.h must compile as C, the library must load with dlopen,
 * and the calls that need no GPU -- version, error strings, parameter validation, the slab partition and message plan --
 * must behave as the header says.  Built and run by tests/test_library_abi.py. */
#include <dlfcn.h>
#include <stdio.h>
#include <string.h>
#include "../../include/smcx.h"

#define CHECK(cond) do { if (!(cond)) { printf("FAILED: %s (line %d)\n", #cond, __LINE__); return 1; } } while (0)

int main(int argc, char **argv) {
  if (argc < 2) { printf("usage: abi_from_c libsmcx.so\n"); return 2; }
  void *lib = dlopen(argv[1], RTLD_NOW | RTLD_LOCAL);
  if (!lib) { printf("dlopen: %s\n", dlerror()); return 3; }
  const char *(*version)(void) = (const char *(*)(void))dlsym(lib, "smcx_version");
  const char *(*strerr)(int) = (const char *(*)(int))dlsym(lib, "smcx_strerror");
  int (*ws_bytes)(const smcx_params_t *, size_t *) = (int (*)(const smcx_params_t *, size_t *))dlsym(lib, "smcx_workspace_bytes");
  int (*partition)(const smcx_params_t *, int32_t, int32_t, smcx_domain_info_t *) =
      (int (*)(const smcx_params_t *, int32_t, int32_t, smcx_domain_info_t *))dlsym(lib, "smcx_domain_partition");
  int (*plan)(const smcx_params_t *, int32_t, int32_t, int64_t, int64_t, int32_t, smcx_domain_msg_t *, smcx_domain_msg_t *) =
      (int (*)(const smcx_params_t *, int32_t, int32_t, int64_t, int64_t, int32_t, smcx_domain_msg_t *, smcx_domain_msg_t *))
          dlsym(lib, "smcx_domain_plan_messages");
  CHECK(version && strerr && ws_bytes && partition && plan);
  CHECK(strstr(version(), "sm_100a") != NULL);
  CHECK(strcmp(strerr(SMCX_OK), "ok") == 0);

  int32_t epi[2 * 4 * 4];
  uint32_t accept[8] = {0xFFFFFFFFu, 1000u, 100u, 10u, 1u, 0u, 0u, 0u};
  for (int s = 0; s < 2; ++s)
    for (int a = 0; a < 4; ++a)
      for (int b = 0; b < 4; ++b) epi[(s * 4 + a) * 4 + b] = (a + 1) * (b + 1) * (s ? -3 : 5);   /* symmetric */
  smcx_params_t p;
  memset(&p, 0, sizeof p);
  p.lattice = SMCX_BCC;
  p.dims[0] = 16; p.dims[1] = 16; p.dims[2] = 32;
  p.n_species = 4; p.n_shells = 2; p.epi = epi; p.link_cell = 4;
  p.accept = accept; p.accept_len = 8; p.seed = 7;
  size_t bytes = 0;
  CHECK(ws_bytes(&p, &bytes) == SMCX_OK && bytes >= 16u * 16u * 32u * 2u / 4u);
  CHECK(ws_bytes(NULL, &bytes) == SMCX_E_NULL_ARG);
  p.dims[2] = 30;
  CHECK(ws_bytes(&p, &bytes) == SMCX_E_BAD_DIMS);
  p.dims[2] = 32;
  epi[1] += 1;
  CHECK(ws_bytes(&p, &bytes) == SMCX_E_EPI_NOT_SYMMETRIC);
  epi[1] -= 1;

  smcx_domain_info_t a, b;
  CHECK(partition(&p, 2, 0, &a) == SMCX_OK && partition(&p, 2, 1, &b) == SMCX_OK);
  CHECK(a.row_first == 0 && a.row_count == 4 && b.row_first == 4 && b.row_count == 4);
  CHECK(a.ghost == 2 && a.z_layers == 4 * 4 + 3 + 4 && a.lower == 1 && a.upper == 1);
  CHECK(partition(&p, 5, 0, &a) == SMCX_E_BAD_DIMS);          /* four pairs of rows only */
  smcx_domain_msg_t s0, r0, s1, r1;
  for (int phase = 0; phase < 8; ++phase) {
    CHECK(plan(&p, 2, 0, 3, 0, phase, &s0, &r0) == SMCX_OK && plan(&p, 2, 1, 3, 0, phase, &s1, &r1) == SMCX_OK);
    CHECK(s0.peer == 1 && s1.peer == 0 && s0.bytes == r1.bytes && s1.bytes == r0.bytes && s0.tag == r1.tag);
    CHECK(s0.bytes == 3 * b.layer_bytes);
  }
  CHECK(plan(&p, 2, 0, 3, 0, 9, &s0, &r0) == SMCX_E_RANGE);
  printf("abi_from_c ok\n");
  dlclose(lib);
  return 0;
}
