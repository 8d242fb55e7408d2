/* zmc_kernel_probe.cu -- a measurement tool, NOT part of the product ABI (like zmc_microbench.cu): ONE level-1 launch of
 * zmc_sample_kernel<ZmcIntegrand<TID, TD, TPREC, TMODE>, TUKEY> on synthetic parents, timed with CUDA events (best of `reps`), with
 * the fraction of the ALU roof and an XOR checksum over all per-(cell, trial) sums, so that variants of the
 * kernel (the ZMC_TUNE_* macros of zmc_device.cuh, ZMC_PACKED_EXP_POLY, ZMC_RANGE_PROOF) can be compared and shown to differ in
 * schedule only. Built and run by `python -m paper_1902_07916_b200.microbench --probe ...`; profiles/r2_pipe_split.md quotes it.
 *   argv: n_instances  divisions_per_axis  samples_per_cell  trials  reps
 *   -DTD=<dim> -DTID=<integrand id> -DTUKEY=<0|1> [-DTMODE=1] [-DTPREC=0] [-DTA=<a of EXP_QUAD at D >= 9>] [-DZMC_TUNE_...=..] */
#include <cstdio>
#include <cstdlib>
#include <vector>
#include <cuda_runtime.h>
#include "zmc_device.cuh"
#ifndef TMODE
#define TMODE 0
#endif
#ifndef TA
#define TA 5000.0
#endif
#ifndef TPREC
#define TPREC 1
#endif
using F = ZmcIntegrand<TID, TD, TPREC, TMODE>;
#define CK(x) do { cudaError_t e = (x); if (e != cudaSuccess) { printf("%s: %s\n", #x, cudaGetErrorString(e)); exit(1); } } while (0)
int main(int argc, char** argv) {
    const int n_inst = argc > 1 ? atoi(argv[1]) : 256;
    const int g = argc > 2 ? atoi(argv[2]) : 6;
    const unsigned long long N = argc > 3 ? atoll(argv[3]) : 4096;
    const int T = argc > 4 ? atoi(argv[4]) : 5;
    const int reps = argc > 5 ? atoi(argv[5]) : 5;
    const int D = TD;
    unsigned long long k = 1;
    for (int d = 0; d < D; ++d) k *= g;
    const unsigned long long n_cells = k * n_inst;
    const int SG = ZmcGroup<TD>::SG;
    ZmcLevelInfo li = {};
    li.n_groups = n_inst; li.n_cells = n_cells; li.n_chunks = 1; li.chunk_groups = (unsigned)((N + SG - 1) / SG);
    const bool tl = ZmcTune<F>::TRIAL_LOOP && n_cells >= 65536;
    li.trials_per_item = tl ? T : 1;
    li.n_items = n_cells * (T / li.trials_per_item);
    ZmcLevelInfo* d_info; CK(cudaMalloc(&d_info, sizeof li));
    std::vector<zu32> inst(n_inst), phi(n_inst, 0), coord((size_t)n_inst * D, 0), keys(2 * n_inst);
    std::vector<zu64> plo(n_inst, 0);
    const int ppi = 2 + D;
    std::vector<double> par((size_t)n_inst * ppi);
    std::vector<float> parf((size_t)n_inst * ppi);
    srand(7);
    for (int i = 0; i < n_inst; ++i) {
        inst[i] = i; keys[2 * i] = rand() * 2654435761u; keys[2 * i + 1] = rand() * 40503u + 17;
        par[(size_t)i * ppi] = 1.0; par[(size_t)i * ppi + 1] = (TID == 3) ? (TD >= 9 ? TA : 1.0 + (i % 100) * 7.0) : 1.0;
        for (int d = 0; d < D; ++d) par[(size_t)i * ppi + 2 + d] = (TD >= 9) ? 0.0 : 0.2 + 0.6 * ((i * 31 + d * 7) % 97) / 97.0;
        for (int j = 0; j < ppi; ++j) parf[(size_t)i * ppi + j] = (float)par[(size_t)i * ppi + j];
    }
    zu32 *d_inst, *d_phi, *d_coord, *d_keys; zu64* d_plo; double *d_par, *d_partial; float* d_parf;
    CK(cudaMalloc(&d_inst, 4 * n_inst)); CK(cudaMalloc(&d_phi, 4 * n_inst)); CK(cudaMalloc(&d_coord, 4 * (size_t)n_inst * D));
    CK(cudaMalloc(&d_keys, 8 * n_inst)); CK(cudaMalloc(&d_plo, 8 * n_inst)); CK(cudaMalloc(&d_par, 8 * par.size())); CK(cudaMalloc(&d_parf, 4 * par.size()));
    CK(cudaMalloc(&d_partial, 8 * n_cells * T));
    CK(cudaMemcpy(d_inst, inst.data(), 4 * n_inst, cudaMemcpyHostToDevice)); CK(cudaMemcpy(d_phi, phi.data(), 4 * n_inst, cudaMemcpyHostToDevice));
    CK(cudaMemcpy(d_coord, coord.data(), 4 * (size_t)n_inst * D, cudaMemcpyHostToDevice)); CK(cudaMemcpy(d_keys, keys.data(), 8 * n_inst, cudaMemcpyHostToDevice));
    CK(cudaMemcpy(d_plo, plo.data(), 8 * n_inst, cudaMemcpyHostToDevice)); CK(cudaMemcpy(d_par, par.data(), 8 * par.size(), cudaMemcpyHostToDevice));
    CK(cudaMemcpy(d_parf, parf.data(), 4 * par.size(), cudaMemcpyHostToDevice));
    ZmcSampleArgs a = {};
    a.par_inst = d_inst; a.par_plo = d_plo; a.par_phi = d_phi; a.par_coord = d_coord; a.par_stride = n_inst; a.info = d_info;
    a.partial = d_partial; a.keys = d_keys; a.params = d_par; a.params_f32 = d_parf; a.ppi = ppi; a.g = g; a.T = T; a.level = 1; a.k = k; a.N = N;
    const double lo = (TD >= 9) ? -1.0 : 0.0, up = (TID == 2) ? 10.0 : 1.0;
    for (int d = 0; d < D; ++d) { a.lower[d] = lo; a.width[d] = (up - lo) / g; }
    a.ukey[0] = keys[0]; a.ukey[1] = keys[1];
    auto kern = zmc_sample_kernel<F, TUKEY != 0, false>;
    cudaFuncAttributes fa; CK(cudaFuncGetAttributes(&fa, kern));
    int per_sm = 0; CK(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, ZMC_BLOCK_THREADS, 0));
    int sms = 0; CK(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, 0));
    const int grid = sms * per_sm;
    cudaEvent_t e0, e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
    float best = 1e30f;
    for (int r = 0; r < reps + 1; ++r) {
        CK(cudaMemcpy(d_info, &li, sizeof li, cudaMemcpyHostToDevice));
        cudaEventRecord(e0);
        kern<<<grid, ZMC_BLOCK_THREADS>>>(a);
        cudaEventRecord(e1);
        CK(cudaEventSynchronize(e1));
        float ms; cudaEventElapsedTime(&ms, e0, e1);
        if (r > 0 && ms < best) best = ms;
    }
    std::vector<double> part(n_cells * T);
    CK(cudaMemcpy(part.data(), d_partial, 8 * part.size(), cudaMemcpyDeviceToHost));
    unsigned long long x = 0; double sum = 0;
    for (size_t i = 0; i < part.size(); ++i) { unsigned long long b; memcpy(&b, &part[i], 8); x ^= b * (2 * i + 1); sum += part[i]; }
    const double evals = (double)n_cells * T * N;
    const double roof = sms * 1.965e9 * 32.0 / (20.0 * D / 4.0);
    printf("D=%d ID=%d UKEY=%d regs=%d ctas/sm=%d grid=%d  %.3f ms  %.4e evals/s  frac %.4f  checksum %016llx sum %.9e\n", D, TID, TUKEY, fa.numRegs, per_sm,
           grid, best, evals / (best * 1e-3), evals / (best * 1e-3) / roof, x, sum);
    return 0;
}
