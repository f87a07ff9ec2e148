// ccl_ubench.cu -- microbenchmark behind the constants in DESIGN.md section 6: throughput of random 4-byte loads,
// atomicMin (with return) and red.min (no return) into an int32 array of 8 MiB ... 1 GiB, with indices streamed
// from a 512 MB array, plus the index stream alone.  Standalone program (no library code); build and run with
//     python -m paper_1603_08357_b200.build --ubench && ./paper_1603_08357_b200/ccl_ubench.bin
#include <cuda_runtime.h>
#include <cstdio>
#include <cstdint>
#include <cstdlib>
#define CK(x) do{cudaError_t e=(x); if(e!=cudaSuccess){printf("ERR %s line %d\n",cudaGetErrorString(e),__LINE__); exit(1);} }while(0)

__device__ __forceinline__ uint32_t hash32(uint32_t x){ x^=x>>16; x*=0x7feb352dU; x^=x>>15; x*=0x846ca68bU; x^=x>>16; return x; }

__global__ void k_fill_idx(int* idx, size_t n, uint32_t mask, uint32_t salt){
  size_t i = blockIdx.x*(size_t)blockDim.x+threadIdx.x; size_t st=(size_t)gridDim.x*blockDim.x;
  for(;i<n;i+=st) idx[i] = hash32((uint32_t)i*2654435761u + salt) & mask;
}
__global__ void k_iota(int* a, size_t n){ size_t i = blockIdx.x*(size_t)blockDim.x+threadIdx.x; size_t st=(size_t)gridDim.x*blockDim.x; for(;i<n;i+=st) a[i]=(int)i; }

// mode 0: ld default; 1: ld.cg (relaxed gpu); 2: atomicMin returning; 3: red (no return); 4: stream only
template<int MODE, int U>
__global__ void __launch_bounds__(256) k_gather(const int* __restrict__ idx, size_t n, int* arr, unsigned long long* out){
  size_t t = blockIdx.x*(size_t)blockDim.x+threadIdx.x;
  size_t base = t*(size_t)(4*U);
  if (base + 4*U > n) return;
  int acc=0;
  int4 v[U];
  #pragma unroll
  for(int u=0;u<U;u++) v[u] = __ldcs(reinterpret_cast<const int4*>(idx+base)+u);
  int r[4*U];
  #pragma unroll
  for(int u=0;u<U;u++){
    int ii[4]={v[u].x,v[u].y,v[u].z,v[u].w};
    #pragma unroll
    for(int k=0;k<4;k++){
      if(MODE==0) r[4*u+k]=arr[ii[k]];
      else if(MODE==1) r[4*u+k]=__ldcg(arr+ii[k]);
      else if(MODE==2) r[4*u+k]=atomicMin(arr+ii[k], ii[k]>>1);
      else if(MODE==3){ atomicMin(arr+ii[k], ii[k]>>1); r[4*u+k]=0; }
      else r[4*u+k]=ii[k];
    }
  }
  #pragma unroll
  for(int j=0;j<4*U;j++) acc^=r[j];
  if(acc==0x7fffffff) out[0]=acc;
}

template<int MODE,int U>
float run(const int* idx, size_t n, int* arr, unsigned long long* out, int reps){
  size_t threads = n/(4*U); int blocks=(int)((threads+255)/256);
  cudaEvent_t a,b; cudaEventCreate(&a); cudaEventCreate(&b);
  k_gather<MODE,U><<<blocks,256>>>(idx,n,arr,out); CK(cudaDeviceSynchronize());
  cudaEventRecord(a);
  for(int r=0;r<reps;r++) k_gather<MODE,U><<<blocks,256>>>(idx,n,arr,out);
  cudaEventRecord(b); CK(cudaDeviceSynchronize());
  float ms; cudaEventElapsedTime(&ms,a,b); return ms/reps;
}

int main(){
  const size_t NIDX = (size_t)1<<27;       // 128M random indices (512 MB stream)
  int* idx; CK(cudaMalloc(&idx,NIDX*4));
  unsigned long long* out; CK(cudaMalloc(&out,8));
  const char* names[5]={"ld.ca","ld.cg","atomMin.ret","red.min","stream-only"};
  for(int lg=21; lg<=28; lg+=1){
    size_t N=(size_t)1<<lg; int* arr; CK(cudaMalloc(&arr,N*4));
    k_fill_idx<<<1184,256>>>(idx,NIDX,(uint32_t)(N-1),lg); 
    float ms[5][3];
    for(int m=0;m<5;m++){
      k_iota<<<1184,256>>>(arr,N); CK(cudaDeviceSynchronize());
      #define R(M) if(m==M){ ms[m][0]=run<M,1>(idx,NIDX,arr,out,3); ms[m][1]=run<M,2>(idx,NIDX,arr,out,3); ms[m][2]=run<M,4>(idx,NIDX,arr,out,3);} 
      R(0) R(1) R(2) R(3) R(4)
    }
    for(int m=0;m<5;m++) printf("array 2^%d ints (%zu MiB) %-12s U=1: %.3f ms %.1f G/s | U=2: %.3f ms %.1f G/s | U=4: %.3f ms %.1f G/s\n", lg,(N*4)>>20,names[m],
        ms[m][0], NIDX/ms[m][0]/1e6, ms[m][1], NIDX/ms[m][1]/1e6, ms[m][2], NIDX/ms[m][2]/1e6);
    cudaFree(arr);
  }
  return 0;
}
