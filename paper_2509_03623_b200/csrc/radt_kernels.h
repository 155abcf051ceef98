// radt_kernels.h -- host-callable launchers of the CUDA kernels (internal to the library).
#pragma once
#include "radt_dev.cuh"

cudaError_t radt_launch_setup(const SetupParams &P, const LevelTable &L, const ChanTable &V, cudaStream_t st);
cudaError_t radt_launch_occ_sph(const SetupParams &P, cudaStream_t st);
cudaError_t radt_launch_unpack(const float4 *grad, long long cells, int nbatch, long long batch_stride, float *g_dens,
                               float *g_temp, float *g_vel, cudaStream_t st);
cudaError_t radt_launch_l2(const float *cube, const float *target, double sigma, long long n, float *dl, double *loss,
                           cudaStream_t st);
cudaError_t radt_launch_loss_finish(double *part, double scale, double *loss, cudaStream_t st);
cudaError_t radt_launch_march_fwd(const MarchParams &P, int nbatch, cudaStream_t st);
cudaError_t radt_launch_march_bwd(const MarchParams &P, int nbatch, cudaStream_t st);
cudaError_t radt_launch_march_fwd_win(const MarchParams &P, int nbatch, cudaStream_t st);
cudaError_t radt_launch_march_bwd_win(const MarchParams &P, int nbatch, cudaStream_t st);
cudaError_t radt_run_pipe_peak(int kind, double *ops_per_s, double *clock_mhz);
cudaError_t radt_launch_disk_fwd(const DiskParamsDev &Q, cudaStream_t st);
cudaError_t radt_launch_disk_bwd(const DiskParamsDev &Q, cudaStream_t st);
cudaError_t radt_launch_disk_fwd_static(DiskParamsDev Q, cudaStream_t st);      // scratch inside the library image (radt_disk.cu)
cudaError_t radt_launch_mlp_fwd(const MlpParamsDev &Q, cudaStream_t st);        // radt_mlp_tc.cu (tcgen05)
cudaError_t radt_launch_mlp_bwd(const MlpParamsDev &Q, int nparams, cudaStream_t st);        // radt_mlp_tc_bwd.cu (tcgen05)
