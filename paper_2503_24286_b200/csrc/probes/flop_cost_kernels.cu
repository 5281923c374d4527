// One-line kernels whose SASS gives the FP64 instruction cost of CUDA's exp, log and division on sm_100a
// ("exp/log/pow counted by their SASS instruction cost").  Not part of libpyro; compiled and
// disassembled only to produce profiles/flop_costs.md:
//   nvcc -gencode arch=compute_100a,code=sm_100a -O3 -cubin -o /tmp/flop_cost.cubin paper_2503_24286_b200/csrc/probes/flop_cost_kernels.cu
//   cuobjdump -sass /tmp/flop_cost.cubin
extern "C" __global__ void k_exp(const double *x, double *y) { y[threadIdx.x] = exp(x[threadIdx.x]); }
extern "C" __global__ void k_log(const double *x, double *y) { y[threadIdx.x] = log(x[threadIdx.x]); }
extern "C" __global__ void k_div(const double *x, double *y) { y[threadIdx.x] = x[threadIdx.x] / x[threadIdx.x + 32]; }
extern "C" __global__ void k_pow(const double *x, double *y) { y[threadIdx.x] = pow(x[threadIdx.x], x[threadIdx.x + 32]); }
