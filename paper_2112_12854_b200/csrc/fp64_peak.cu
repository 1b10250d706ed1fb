// fp64_peak.cu -- DFMA microbenchmark behind the "alu" roof of DESIGN.md section 6: dependent-issue latency, ILP scaling and
// full-chip throughput of the plain fp64 pipe on B200.  Build and run (profiles/r01_fp64_peak.md has the output):
//   nvcc -O3 -gencode arch=compute_100a,code=sm_100a -o /tmp/fp64_peak paper_2112_12854_b200/csrc/fp64_peak.cu && /tmp/fp64_peak
#include <cstdio>
#include <cuda_runtime.h>
template<int ILP> __global__ void dfma_chain(double* out, int n, double a, double b, long long* cyc) {
    double x[ILP];
    for (int j=0;j<ILP;++j) x[j] = threadIdx.x*1e-9 + j;
    long long t0 = clock64();
    #pragma unroll 1
    for (int i=0;i<n;++i) {
        #pragma unroll
        for (int r=0;r<8;++r) {
            #pragma unroll
            for (int j=0;j<ILP;++j) x[j] = fma(x[j], a, b);
        }
    }
    long long t1 = clock64();
    double s=0; for (int j=0;j<ILP;++j) s+=x[j];
    out[blockIdx.x*blockDim.x+threadIdx.x]=s;
    if (threadIdx.x==0 && blockIdx.x==0) *cyc = t1-t0;
}
template<int ILP> void run(int blocks, int threads, const char* tag) {
    double* out; long long* cyc; cudaMalloc(&out, sizeof(double)*blocks*threads); cudaMalloc(&cyc, 8);
    int n = 2000;
    dfma_chain<ILP><<<blocks,threads>>>(out,n,0.999999,1e-7,cyc); cudaDeviceSynchronize();
    cudaEvent_t e0,e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
    cudaEventRecord(e0); dfma_chain<ILP><<<blocks,threads>>>(out,n,0.999999,1e-7,cyc); cudaEventRecord(e1); cudaDeviceSynchronize();
    float ms; cudaEventElapsedTime(&ms,e0,e1); long long c; cudaMemcpy(&c,cyc,8,cudaMemcpyDeviceToHost);
    double instr = (double)n*8*ILP;  // per thread
    double total = instr*blocks*threads;
    printf("%s ILP=%d blocks=%d threads=%d: %.2f cycles/DFMA(per warp, block0), %.2f TFLOP/s (fma=2), ms=%.3f\n", tag, ILP, blocks, threads, (double)c/instr, total*2/ms/1e9, ms);
    cudaFree(out); cudaFree(cyc);
}
int main(){
    run<1>(148,32,"1warp/SM"); run<2>(148,32,"1warp/SM"); run<4>(148,32,"1warp/SM"); run<8>(148,32,"1warp/SM");
    run<1>(148,128,"1warp/SMSP"); run<2>(148,128,"1warp/SMSP"); run<4>(148,128,"1warp/SMSP");
    run<1>(148*2,256,"4warp/SMSP"); run<2>(148*2,256,"4warp/SMSP"); run<4>(148*2,256,"4warp/SMSP");
    run<1>(148*2,512,"8warp/SMSP"); run<2>(148*2,512,"8warp/SMSP"); run<4>(148*4,512,"16warp/SMSP");
    return 0;
}
