// microbench_l2_gather.cu -- standalone probe (not part of libpainn_b200.so): L2 -> SM bandwidth for sequential reads and for
// the row-gather pattern of the edge kernels (a warp reads one 512 B or 2 KB row per request, rows picked at random inside
// a window of neighbours).  Its result is the denominator of roofline.l2_gather in bench.py (profiles/r01_microbench.md).
//   nvcc -gencode arch=compute_100a,code=sm_100a -O3 -o /tmp/l2_gather paper_2506_04055_b200/csrc/microbench_l2_gather.cu && /tmp/l2_gather
#include <cstdio>
#include <cstdlib>
#include <cuda_runtime.h>
#include <vector>
#define CK(x) do{cudaError_t e=(x); if(e!=cudaSuccess){printf("err %s line %d\n",cudaGetErrorString(e),__LINE__);exit(1);} }while(0)

__global__ void k_seq(const float4* __restrict__ a, size_t n, int reps, float* out){
  float acc=0; size_t tid=blockIdx.x*(size_t)blockDim.x+threadIdx.x, st=(size_t)gridDim.x*blockDim.x;
  for(int r=0;r<reps;r++) for(size_t i=tid;i<n;i+=st*4){
    float4 v0=a[i], v1=i+st<n?a[i+st]:v0, v2=i+2*st<n?a[i+2*st]:v0, v3=i+3*st<n?a[i+3*st]:v0;
    acc+=v0.x+v1.y+v2.z+v3.w;}
  if(acc==1.2345f) out[0]=acc;
}
// gather: each warp reads ROWB bytes rows (lane -> 16 B * k), idx list; U rows in flight
template<int U, int V4PL> // V4PL float4 per lane per row  (row bytes = 512*V4PL)
__global__ void k_gather(const float4* __restrict__ tab, const int* __restrict__ idx, size_t nidx, float* out){
  const int lane=threadIdx.x&31; size_t w=(blockIdx.x*(size_t)blockDim.x+threadIdx.x)>>5, nw=((size_t)gridDim.x*blockDim.x)>>5;
  float acc=0;
  for(size_t b=w*U;b+U<=nidx;b+=nw*U){
    float4 v[U][V4PL];
    #pragma unroll
    for(int u=0;u<U;u++){ const int r=idx[b+u];
      #pragma unroll
      for(int q=0;q<V4PL;q++) v[u][q]=__ldg(tab+(size_t)r*32*V4PL+q*32+lane);}
    #pragma unroll
    for(int u=0;u<U;u++)
      #pragma unroll
      for(int q=0;q<V4PL;q++) acc+=v[u][q].x+v[u][q].w;
  }
  if(acc==1.2345f) out[0]=acc;
}
int main(){
  int nsm; CK(cudaDeviceGetAttribute(&nsm,cudaDevAttrMultiProcessorCount,0));
  float* out; CK(cudaMalloc(&out,4));
  cudaEvent_t e0,e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
  // sequential, sizes 32MB..4GB
  for(size_t mb: {16,32,64,96,256,2048}){
    size_t n=mb*1024*1024/16; float4* a; CK(cudaMalloc(&a,n*16)); CK(cudaMemset(a,0,n*16));
    int reps= mb<=96? 50: 4;
    for(int bl: {1,2,4,8}){
    k_seq<<<nsm*bl,512>>>(a,n,2,out);
    cudaEventRecord(e0); k_seq<<<nsm*bl,512>>>(a,n,reps,out); cudaEventRecord(e1); CK(cudaDeviceSynchronize());
    float ms; cudaEventElapsedTime(&ms,e0,e1);
    printf("seq %zu MB blocks/SM %d: %.1f GB/s\n",mb,bl,(double)n*16*reps/ms/1e6);}
    cudaFree(a);
  }
  // gather rows: table sizes; locality: random within window
  for(int v4pl: {1,4}){
   for(size_t tabmb: {32, 2048}){
    size_t rowb=512*v4pl, nrows=tabmb*1024*1024/rowb; float4* tab; CK(cudaMalloc(&tab,nrows*rowb)); CK(cudaMemset(tab,0,nrows*rowb));
    for(int window: {400, 0}){
      size_t nidx=(size_t)1<<24; if(v4pl==4) nidx>>=2; std::vector<int> h(nidx);
      for(size_t i=0;i<nidx;i++){ if(window){ size_t c=(i/64)%nrows; long r=(long)c+(rand()%window)-window/2; if(r<0)r+=nrows; h[i]=r%nrows;} else h[i]=((size_t)rand()*RAND_MAX+rand())%nrows; }
      int* idx; CK(cudaMalloc(&idx,nidx*4)); CK(cudaMemcpy(idx,h.data(),nidx*4,cudaMemcpyHostToDevice));
      for(int bl:{2,4,8}){
        auto run=[&](){ if(v4pl==1) k_gather<16,1><<<nsm*bl,256>>>(tab,idx,nidx,out); else k_gather<8,4><<<nsm*bl,256>>>(tab,idx,nidx,out); };
        run(); cudaEventRecord(e0); run(); cudaEventRecord(e1); CK(cudaDeviceSynchronize());
        float ms; cudaEventElapsedTime(&ms,e0,e1);
        printf("gather row %zu B table %zu MB window %d blocks/SM %d: %.1f GB/s\n",rowb,tabmb,window,bl,(double)nidx*rowb/ms/1e6);
      }
      cudaFree(idx);
    }
    cudaFree(tab);
   }
  }
  return 0;
}
