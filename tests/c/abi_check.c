/* Calls the C ABI of include/ent.h from plain C (no Python, no ctypes): create -> set_grid -> error paths -> workspace query.
 * Exit code 0 = every check passed; prints "no device" and exits 0 after the ent_create check when no CUDA device exists
 * (the library has no CPU fallback, so that is the only call that can be exercised there). */
#include <stdio.h>
#include <string.h>
#include "ent.h"

#define CHECK(cond) do { if (!(cond)) { fprintf(stderr, "abi_check: line %d: %s failed (%s)\n", __LINE__, #cond, ctx ? ent_last_error(ctx) : ""); return 1; } } while (0)

int main(void) {
    ent_ctx *ctx = NULL;
    CHECK(ent_version() != NULL && strchr(ent_version(), '.') != NULL);
    CHECK(ent_create(NULL, 0, NULL) == ENT_EINVAL);
    int rc = ent_create(&ctx, 0, NULL);
    if (rc == ENT_ECUDA) { CHECK(ctx == NULL); printf("no device\n"); return 0; }
    CHECK(rc == ENT_OK && ctx != NULL);
    CHECK(strcmp(ent_last_error(ctx), "") == 0);

    ent_grid g;
    memset(&g, 0, sizeof g);
    size_t bytes = 0;
    CHECK(ent_workspace_bytes(ctx, 1000, &bytes) == ENT_EINVAL);          /* no grid yet */
    g.D = 4;
    CHECK(ent_set_grid(ctx, &g) == ENT_EINVAL);                           /* D not in {2,3} */
    g.D = 3; g.N[0] = 16; g.N[1] = 16; g.N[2] = 2; g.kind = ENT_CART;
    for (int a = 0; a < 3; ++a) { g.bc[a] = ENT_PERIODIC; g.xmin[a] = 0.0; g.xmax[a] = 8.0; }
    CHECK(ent_set_grid(ctx, &g) == ENT_EINVAL);                           /* periodic dimension with N < 3 */
    CHECK(strlen(ent_last_error(ctx)) > 0);
    g.N[2] = 16;
    g.xmax[1] = -1.0;
    CHECK(ent_set_grid(ctx, &g) == ENT_EINVAL);                           /* xmax <= xmin */
    g.xmax[1] = 8.0;
    g.kind = ENT_SPH;
    CHECK(ent_set_grid(ctx, &g) == ENT_EUNSUPPORTED);                     /* SPH needs D == 2 */
    g.kind = ENT_CART; g.bc[0] = ENT_AXIS;
    CHECK(ent_set_grid(ctx, &g) == ENT_EUNSUPPORTED);                     /* AXIS on a Cartesian grid */
    g.bc[0] = ENT_PERIODIC;
    CHECK(ent_set_grid(ctx, &g) == ENT_OK);

    int64_t v = 0;
    CHECK(ent_get_stat(ctx, ENT_STAT_TILE_1, &v) == ENT_OK && v == 8);
    CHECK(ent_get_stat(ctx, ENT_STAT_NTILES, &v) == ENT_OK && v == 8);
    CHECK(ent_get_stat(ctx, ENT_STAT_NKEYS, &v) == ENT_OK && v == 4096);
    CHECK(ent_get_stat(ctx, 999, &v) == ENT_EINVAL);
    CHECK(ent_set_option(ctx, ENT_OPT_STEP_IMPL, 7) == ENT_EINVAL);
    CHECK(ent_workspace_bytes(ctx, 100000, &bytes) == ENT_OK && bytes > 100000u * 4u);
    size_t bytes2 = 0;
    CHECK(ent_workspace_bytes(ctx, 200000, &bytes2) == ENT_OK && bytes2 > bytes);
    CHECK(ent_reserve(ctx, 100000) == ENT_OK);
    CHECK(ent_get_stat(ctx, ENT_STAT_SCRATCH_BYTES, &v) == ENT_OK && (size_t)v == bytes);

    /* NULL / misaligned arguments are refused before anything is launched */
    ent_fields F; ent_current J; ent_particles p;
    memset(&F, 0, sizeof F); memset(&J, 0, sizeof J); memset(&p, 0, sizeof p);
    int64_t launches = 0, launches2 = 0;
    CHECK(ent_get_stat(ctx, ENT_STAT_LAUNCHES, &launches) == ENT_OK);
    CHECK(ent_step(ctx, &F, &p, &J, 0.1f) == ENT_EINVAL);                 /* NULL field arrays */
    CHECK(ent_step(ctx, NULL, &p, &J, 0.1f) == ENT_EINVAL);
    CHECK(ent_sort(ctx, NULL, &p, NULL) == ENT_EINVAL);
    CHECK(ent_step_sorted(ctx, &F, &p, &p, &J, 0.1f) == ENT_EINVAL);
    CHECK(ent_forget(ctx, NULL) == ENT_EINVAL);
    p.n = -5;
    CHECK(ent_gather_push(ctx, &F, &p, &p, 0.1f) == ENT_EINVAL);
    CHECK(ent_get_stat(ctx, ENT_STAT_LAUNCHES, &launches2) == ENT_OK && launches2 == launches);
    CHECK(ent_destroy(ctx) == ENT_OK);
    CHECK(ent_destroy(NULL) == ENT_EINVAL);
    printf("abi ok\n");
    return 0;
}
