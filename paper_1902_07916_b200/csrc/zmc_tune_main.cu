/*
 * zmc_tune_main.cu -- stand-alone timing of one instance of zmc_sample_kernel (python -m paper_1902_07916_b200.tune).
 *
 * One level-1 launch of a synthetic workload of the given dimension through the committed device header, compiled with
 * -DZMC_TUNE_PACKED / _UNROLL / _MINB / _P0ADD overrides of ZmcTune; prints time, evaluations/s, the fraction of the
 * IMAD.WIDE roof and an XOR checksum over all per-(cell, trial) sums: every variant of a case must
 * print the same checksum (the variants differ in schedule, never in arithmetic).
 * -DVD=<dim> -DVID=<integrand id> -DVMODE=<0 exact | 1 fast> -DVUKEY=<true|false> -DVSQ=<true|false> -DVNAME="..."
 */
#include <cuda_runtime.h>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <vector>
#include "zmc_device.cuh"

#ifndef VD
#define VD 6
#endif
#ifndef VID
#define VID ZMC_ID_SIN_SUM
#endif
#ifndef VMODE
#define VMODE ZMC_MODE_EXACT
#endif
#ifndef VUKEY
#define VUKEY true
#endif
#ifndef VSQ
#define VSQ false
#endif
#ifndef VNAME
#define VNAME "base"
#endif

#define CK(x) do { cudaError_t e_ = (x); if (e_ != cudaSuccess) { printf("CUDA error %s at %d\n", cudaGetErrorString(e_), __LINE__); exit(1); } } while (0)

int main(int argc, char** argv) {
    const int D = VD;
    int g = (VD == 6) ? 4 : 3;
    zu64 N = (VD == 6) ? 100000 : 20000;
    int T = 5;
    if (VD == 4) { g = 6; N = 4096 * 16; }
    if (VD == 12) { g = 2; N = 20000; }
    zu64 k = 1;
    for (int d = 0; d < D; ++d) k *= g;
    typedef ZmcIntegrand<VID, VD, ZMC_PREC_F32, VMODE> F;
    constexpr int SG = ZmcGroup<VD>::SG;

    ZmcSampleArgs a;
    memset(&a, 0, sizeof(a));
    zu32 h_inst = 0; zu64 h_plo = 0; zu32 h_phi = 0;
    std::vector<zu32> h_coord(D, 0);
    zu32 *d_inst, *d_phi, *d_coord, *d_keys; zu64* d_plo; double* d_params; float* d_paramsf; double* d_partial; ZmcLevelInfo* d_info;
    CK(cudaMalloc(&d_inst, 4)); CK(cudaMalloc(&d_phi, 4)); CK(cudaMalloc(&d_plo, 8)); CK(cudaMalloc(&d_coord, 4 * D));
    CK(cudaMalloc(&d_keys, 8)); CK(cudaMalloc(&d_params, 8 * 32)); CK(cudaMalloc(&d_paramsf, 4 * 32));
    CK(cudaMemcpy(d_inst, &h_inst, 4, cudaMemcpyHostToDevice)); CK(cudaMemcpy(d_phi, &h_phi, 4, cudaMemcpyHostToDevice));
    CK(cudaMemcpy(d_plo, &h_plo, 8, cudaMemcpyHostToDevice)); CK(cudaMemcpy(d_coord, h_coord.data(), 4 * D, cudaMemcpyHostToDevice));
    zu32 keys[2] = {0x12345678u, 0x9abcdef0u};
    CK(cudaMemcpy(d_keys, keys, 8, cudaMemcpyHostToDevice));
    double params[32] = {0};
    double lower = 0.0, upper = 10.0;
    if (VID == ZMC_ID_EXP_QUAD) { params[0] = 1.0; params[1] = 5000.0; lower = -1.0; upper = 1.0; if (VD == 4) { params[1] = 30.0; lower = 0; upper = 1; for (int d = 0; d < D; ++d) params[2 + d] = 0.4; } }
    float paramsf[32];
    for (int i = 0; i < 32; ++i) paramsf[i] = (float)params[i];
    CK(cudaMemcpy(d_params, params, sizeof(params), cudaMemcpyHostToDevice));
    CK(cudaMemcpy(d_paramsf, paramsf, sizeof(paramsf), cudaMemcpyHostToDevice));
    const zu64 n_items = k * T;
    CK(cudaMalloc(&d_partial, 8 * n_items));
    double* d_partial_q = nullptr;
    CK(cudaMalloc(&d_partial_q, 8 * n_items));
    CK(cudaMalloc(&d_info, sizeof(ZmcLevelInfo)));
    ZmcLevelInfo li;
    memset(&li, 0, sizeof(li));
    li.n_groups = 1; li.n_cells = k; li.n_items = n_items; li.n_chunks = 1; li.chunk_groups = (zu32)((N + SG - 1) / SG);
    a.par_inst = d_inst; a.par_plo = d_plo; a.par_phi = d_phi; a.par_coord = d_coord; a.par_stride = 1; a.info = d_info;
    a.partial = d_partial; a.partial_q = d_partial_q; a.keys = d_keys; a.params = d_params; a.params_f32 = d_paramsf; a.ppi = 2 + D;
    a.ukey[0] = keys[0]; a.ukey[1] = keys[1]; a.g = g; a.T = T; a.level = 1; a.k = k; a.N = N;
    for (int d = 0; d < D; ++d) { a.lower[d] = lower; a.width[d] = (upper - lower) / g; }

    int dev = 0, sms = 0, occ = 0;
    CK(cudaGetDevice(&dev));
    CK(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    CK(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, zmc_sample_kernel<F, VUKEY, VSQ>, ZMC_BLOCK_THREADS, 0));
    cudaFuncAttributes fa;
    CK(cudaFuncGetAttributes(&fa, zmc_sample_kernel<F, VUKEY, VSQ>));
    const int grid = sms * occ;
    cudaEvent_t e0, e1;
    CK(cudaEventCreate(&e0)); CK(cudaEventCreate(&e1));
    float best = 1e30f;
    for (int rep = 0; rep < 6; ++rep) {
        CK(cudaMemcpy(d_info, &li, sizeof(li), cudaMemcpyHostToDevice));
        CK(cudaEventRecord(e0));
        zmc_sample_kernel<F, VUKEY, VSQ><<<grid, ZMC_BLOCK_THREADS>>>(a);
        CK(cudaEventRecord(e1));
        CK(cudaEventSynchronize(e1));
        float ms;
        CK(cudaEventElapsedTime(&ms, e0, e1));
        if (rep > 0 && ms < best) best = ms;
    }
    std::vector<double> h(n_items);
    CK(cudaMemcpy(h.data(), d_partial, 8 * n_items, cudaMemcpyDeviceToHost));
    unsigned long long x = 0; double sum = 0;
    for (zu64 i = 0; i < n_items; ++i) { unsigned long long b; memcpy(&b, &h[i], 8); x ^= b * (2 * i + 1); sum += h[i]; }
    const double evals = (double)n_items * (double)N;
    const double peak = sms * 1965e6 * 32.0 / (20.0 * D / 4.0);
    printf("%-28s D=%d id=%d mode=%d regs=%d occ=%d thr=%d  %.3f ms  %.2f Gevals/s  frac=%.3f  chk=%016llx sum=%.10g\n", VNAME, D, VID, VMODE,
           fa.numRegs, occ, ZMC_BLOCK_THREADS, best, evals / best * 1e-6, evals / (best * 1e-3) / peak, x, sum);
    return 0;
}
