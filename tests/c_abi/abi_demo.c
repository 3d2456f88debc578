/* abi_demo.c — libwri through its C ABI alone (include/wri.h): plain C99, the CUDA runtime for device
 * memory, no Python and no torch.  Reads one problem from a binary file, runs wri_apply_M,
 * wri_lsqr_batch and wri_objective_gradient_static, writes the results to another file;
 * tests/test_gpu_c_abi.py generates the inputs, builds and runs this program and compares the results
 * with the CPU oracle.
 *
 * input  : int32 nx ny nz nb n_rec L maxit n_omega | double h lambda | double omega[n_omega]
 *          | int32 omega_idx[nb] | int32 rec_ijk[n_rec][3] | float m[n_g] | c64 q[n_g][nb] | c64 d[n_rec][nb]
 * output : c64 ytop[n_g][nb] | c64 ybot[n_rec][nb] | c64 u[n_g][nb] | float resnorms[maxit+1][nb] | int32 iters[nb]
 *          | double f_pde[nb] | double f_data[nb] | float g[n_g]
 */
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>
#include <stdlib.h>

#include "../../include/wri.h"

#define CHECK(x)                                                                         \
    do {                                                                                 \
        int rc__ = (x);                                                                  \
        if (rc__ != 0) {                                                                 \
            fprintf(stderr, "%s failed: %d (%s)\n", #x, rc__, wri_strerror(rc__));       \
            return 2;                                                                    \
        }                                                                                \
    } while (0)
#define CU(x)                                                                            \
    do {                                                                                 \
        cudaError_t e__ = (x);                                                           \
        if (e__ != cudaSuccess) {                                                        \
            fprintf(stderr, "%s failed: %s\n", #x, cudaGetErrorString(e__));             \
            return 3;                                                                    \
        }                                                                                \
    } while (0)

static int rd(void* p, size_t n, FILE* f) { return fread(p, 1, n, f) == n ? 0 : 1; }

int main(int argc, char** argv) {
    if (argc != 3) return 1;
    FILE* f = fopen(argv[1], "rb");
    if (!f) return 1;
    int32_t hd[8];
    double hl[2];
    if (rd(hd, sizeof hd, f) || rd(hl, sizeof hl, f)) return 1;
    const int nx = hd[0], ny = hd[1], nz = hd[2], nb = hd[3], n_rec = hd[4], L = hd[5], maxit = hd[6], n_om = hd[7];
    const size_t ng = (size_t)nx * ny * nz, vb = ng * nb * 8, db = (size_t)n_rec * nb * 8;
    double* omega = malloc(n_om * sizeof(double));
    int32_t* oi = malloc(nb * sizeof(int32_t));
    int32_t* rec = malloc((size_t)n_rec * 3 * sizeof(int32_t));
    float* m = malloc(ng * sizeof(float));
    void *q = malloc(vb), *d = malloc(db);
    if (rd(omega, n_om * sizeof(double), f) || rd(oi, nb * sizeof(int32_t), f) ||
        rd(rec, (size_t)n_rec * 3 * sizeof(int32_t), f) || rd(m, ng * sizeof(float), f) || rd(q, vb, f) || rd(d, db, f))
        return 1;
    fclose(f);

    float* m_dev;
    void *q_dev, *d_dev, *ytop_dev, *ybot_dev, *u_dev, *ws_dev;
    float* res_dev;
    int32_t* it_dev;
    CU(cudaMalloc((void**)&m_dev, ng * sizeof(float)));
    CU(cudaMalloc(&q_dev, vb)); CU(cudaMalloc(&d_dev, db)); CU(cudaMalloc(&ytop_dev, vb));
    CU(cudaMalloc(&ybot_dev, db)); CU(cudaMalloc(&u_dev, vb));
    CU(cudaMalloc((void**)&res_dev, (size_t)(maxit + 1) * nb * sizeof(float)));
    CU(cudaMalloc((void**)&it_dev, nb * sizeof(int32_t)));
    CU(cudaMemcpy(m_dev, m, ng * sizeof(float), cudaMemcpyHostToDevice));
    CU(cudaMemcpy(q_dev, q, vb, cudaMemcpyHostToDevice));
    CU(cudaMemcpy(d_dev, d, db, cudaMemcpyHostToDevice));

    wri_ctx* ctx = NULL;
    wri_grid grid = {nx, ny, nz};
    wri_sponge sp = {L, 1.0f, 2, 0x3Fu};
    CHECK(wri_create(&ctx, grid, hl[0], n_om, omega, m_dev, sp, n_rec, rec, nb, NULL));
    const size_t wsb = wri_workspace_bytes(ctx, nb, 0);
    CU(cudaMalloc(&ws_dev, wsb));
    CHECK(wri_set_workspace(ctx, ws_dev, wsb));
    CHECK(wri_apply_M(ctx, nb, oi, (float)hl[1], q_dev, ytop_dev, ybot_dev));
    CHECK(wri_lsqr_batch(ctx, nb, oi, q_dev, d_dev, (float)hl[1], NULL, maxit, u_dev, res_dev, it_dev));
    CU(cudaDeviceSynchronize());
    /* error behaviour: a too small workspace is refused, not crashed on */
    CHECK(wri_set_workspace(ctx, ws_dev, 16));
    if (wri_lsqr_batch(ctx, nb, oi, q_dev, d_dev, (float)hl[1], NULL, maxit, u_dev, res_dev, it_dev) != WRI_ERR_WORKSPACE)
        return 4;

    /* objective and gradient at the solve's u through the entry that needs neither a workspace (the
     * 16-byte one is still set) nor any device allocation of its own: outputs allocated here, before */
    double *fp_dev = NULL, *fd_dev = NULL;
    float* g_dev = NULL;
    CU(cudaMalloc((void**)&fp_dev, nb * sizeof(double))); CU(cudaMalloc((void**)&fd_dev, nb * sizeof(double)));
    CU(cudaMalloc((void**)&g_dev, ng * sizeof(float)));
    CU(cudaMemset(g_dev, 0, ng * sizeof(float)));
    CHECK(wri_objective_gradient_static(ctx, nb, oi, NULL, NULL, q_dev, u_dev, d_dev, (float)hl[1], fp_dev, fd_dev, g_dev));
    CU(cudaDeviceSynchronize());
    double *fp = malloc(nb * sizeof(double)), *fd = malloc(nb * sizeof(double));
    float* g = malloc(ng * sizeof(float));
    CU(cudaMemcpy(fp, fp_dev, nb * sizeof(double), cudaMemcpyDeviceToHost));
    CU(cudaMemcpy(fd, fd_dev, nb * sizeof(double), cudaMemcpyDeviceToHost));
    CU(cudaMemcpy(g, g_dev, ng * sizeof(float), cudaMemcpyDeviceToHost));

    void *ytop = malloc(vb), *ybot = malloc(db), *u = malloc(vb);
    float* res = malloc((size_t)(maxit + 1) * nb * sizeof(float));
    int32_t* it = malloc(nb * sizeof(int32_t));
    CU(cudaMemcpy(ytop, ytop_dev, vb, cudaMemcpyDeviceToHost));
    CU(cudaMemcpy(ybot, ybot_dev, db, cudaMemcpyDeviceToHost));
    CU(cudaMemcpy(u, u_dev, vb, cudaMemcpyDeviceToHost));
    CU(cudaMemcpy(res, res_dev, (size_t)(maxit + 1) * nb * sizeof(float), cudaMemcpyDeviceToHost));
    CU(cudaMemcpy(it, it_dev, nb * sizeof(int32_t), cudaMemcpyDeviceToHost));
    f = fopen(argv[2], "wb");
    if (!f) return 1;
    fwrite(ytop, 1, vb, f); fwrite(ybot, 1, db, f); fwrite(u, 1, vb, f);
    fwrite(res, sizeof(float), (size_t)(maxit + 1) * nb, f); fwrite(it, sizeof(int32_t), nb, f);
    fwrite(fp, sizeof(double), nb, f); fwrite(fd, sizeof(double), nb, f); fwrite(g, sizeof(float), ng, f);
    fclose(f);
    printf("launches %lld\n", (long long)wri_launch_count(ctx));
    CHECK(wri_destroy(ctx));
    return 0;
}
