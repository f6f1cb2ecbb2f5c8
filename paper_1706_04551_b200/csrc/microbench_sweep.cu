// microbench_sweep.cu -- standalone microbenchmark of the "marching warps" access pattern of
// nh_solver.cu on empty planes: what does the bare traffic pattern of a solver pass cost on this GPU?
// (DESIGN.md section 6 quotes its numbers; profiles/r01i_microbench.md holds one output.)
//
//   nvcc -std=c++17 -O3 -gencode arch=compute_100a,code=sm_100a --extended-lambda \
//        -o microbench_sweep paper_1706_04551_b200/csrc/microbench_sweep.cu
//   ./microbench_sweep [n = 8192] [lead = 4]
//
// n x n cells -> (n+1)^2 nodes in planes laid out like the solver's (60-column strips, `lead` padding
// columns on the left: 4 = strips start on 32-byte sectors, 2 = the earlier 16-byte offset).  Each
// variant reads NL planes and writes NS planes per row (one 16-byte access per lane per plane), with
// the loads of a row issued up front (PF = 0) or one row ahead (PF = 1), plain or streaming (CS)
// stores.  Not part of the library; shares only the geometry constants with it by restating them.
#include <cstdio>
#include <cstdlib>
#include <cuda_runtime.h>
#define CK(x) do{cudaError_t e=(x); if(e!=cudaSuccess){printf("%s:%d %s\n",__FILE__,__LINE__,cudaGetErrorString(e)); exit(1);} }while(0)
constexpr int NT=256, NW=8, SW=60;
struct Pl { double* a[16]; int np, nny, nnx, nstrips, R, nbands; };
__device__ __forceinline__ double2 ld2(const double* a, size_t k){ return *reinterpret_cast<const double2*>(a+k); }
__device__ __forceinline__ void st2(double* a, size_t k, double2 v){ *reinterpret_cast<double2*>(a+k)=v; }
__device__ __forceinline__ void st2cs(double* a, size_t k, double2 v){ __stcs(reinterpret_cast<double2*>(a+k), v); }
// NL loads, NS stores per row; PF: prefetch next row (ping-pong); CS: streaming stores
template<int NL,int NS,int PF,int CS>
__global__ void __launch_bounds__(NT,2) k_sweep(Pl P, double* out){
  const int lane=threadIdx.x&31; const int gw=blockIdx.x*NW+(threadIdx.x>>5), tw=gridDim.x*NW;
  const int nunits=P.nstrips*P.nbands; double acc=0;
  for(int u=gw;u<nunits;u+=tw){
    int strip=u%P.nstrips, band=u/P.nstrips; int c0=strip*SW-2+2*lane; int Ja=band*P.R, Jb=min(Ja+P.R,P.nny);
    bool own=(lane>=1&&lane<=30)&&c0+1<P.nnx;
    double2 A[NL>0?NL:1], B[NL>0?NL:1];
    auto load=[&](double2* X,int j){ size_t k=(size_t)j*P.np+c0; _Pragma("unroll") for(int i=0;i<NL;++i) X[i]=ld2(P.a[i],k); };
    auto step=[&](int j,double2* cur,double2* nxt){
      if(PF) load(nxt,min(j+1,Jb-1)); else load(cur,j);
      double2 s=make_double2(1.0,2.0);
      _Pragma("unroll") for(int i=0;i<NL;++i){ s.x=fma(s.x,1.0000001,cur[i].x); s.y=fma(s.y,0.9999999,cur[i].y);} 
      double w=__shfl_up_sync(0xffffffffu,s.y,1), e=__shfl_down_sync(0xffffffffu,s.x,1);
      s.x+=w*1e-9; s.y+=e*1e-9;
      size_t k=(size_t)j*P.np+c0;
      if(own){ _Pragma("unroll") for(int i=0;i<NS;++i){ double2 v=make_double2(s.x+i,s.y-i); if(CS) st2cs(P.a[10+i],k,v); else st2(P.a[10+i],k,v);} }
      acc+=s.x+s.y;
    };
    if(PF) load(A,Ja);
    for(int j=Ja;j<Jb;j+=2){ step(j,A,B); if(j+1<Jb) step(j+1,B,A); }
  }
  if(acc==123.456) out[0]=acc;
}
template<int NL,int NS,int PF,int CS>
void run(const char* name, Pl P, double* out, size_t nodes){
  cudaEvent_t e0,e1; CK(cudaEventCreate(&e0)); CK(cudaEventCreate(&e1));
  int occ=0; CK(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ,k_sweep<NL,NS,PF,CS>,NT,0));
  int grid=occ*148;
  for(int i=0;i<2;++i) k_sweep<NL,NS,PF,CS><<<grid,NT>>>(P,out);
  CK(cudaEventRecord(e0)); const int reps=10;
  for(int i=0;i<reps;++i) k_sweep<NL,NS,PF,CS><<<grid,NT>>>(P,out);
  CK(cudaEventRecord(e1)); CK(cudaDeviceSynchronize()); float ms; CK(cudaEventElapsedTime(&ms,e0,e1)); ms/=reps;
  double gb=(double)(NL+NS)*8.0*nodes/1e9;
  printf("%-28s NL=%2d NS=%d PF=%d CS=%d occ=%d  %8.1f us  %7.1f GB/s (alg)\n",name,NL,NS,PF,CS,occ,ms*1e3,gb/(ms*1e-3));
}
__global__ void __launch_bounds__(256) k_flat_set(double2* a, size_t n2, double v){ size_t st=(size_t)gridDim.x*blockDim.x; for(size_t k=(size_t)blockIdx.x*blockDim.x+threadIdx.x;k<n2;k+=st) a[k]=make_double2(v,v+k); }
__global__ void __launch_bounds__(256) k_flat_copy(const double2* __restrict__ a, double2* __restrict__ b, size_t n2){ size_t st=(size_t)gridDim.x*blockDim.x; for(size_t k=(size_t)blockIdx.x*blockDim.x+threadIdx.x;k<n2;k+=st) b[k]=a[k]; }
__global__ void __launch_bounds__(256) k_flat_read(const double2* __restrict__ a, double* out, size_t n2){ size_t st=(size_t)gridDim.x*blockDim.x; double s=0; for(size_t k=(size_t)blockIdx.x*blockDim.x+threadIdx.x;k<n2;k+=st){ double2 v=a[k]; s+=v.x+v.y;} if(s==1.2345) out[0]=s; }
template<typename F> void timeit(const char* name, double gb, F f){ cudaEvent_t e0,e1; CK(cudaEventCreate(&e0)); CK(cudaEventCreate(&e1)); f(); f(); CK(cudaEventRecord(e0)); for(int i=0;i<10;++i) f(); CK(cudaEventRecord(e1)); CK(cudaDeviceSynchronize()); float ms; CK(cudaEventElapsedTime(&ms,e0,e1)); ms/=10; printf("%-40s %8.1f us %7.1f GB/s\n",name,ms*1e3,gb/(ms*1e-3)); }

int main(int argc,char**argv){
  int n=argc>1?atoi(argv[1]):8192; int nnx=n+1,nny=n+1; int nstrips=(nnx+SW-1)/SW;
  int lead=argc>2?atoi(argv[2]):4; int np=SW*nstrips+4+lead; np=(np+15)/16*16; int rows=nny+5;
  Pl P; P.np=np;P.nny=nny;P.nnx=nnx;P.nstrips=nstrips;
  int tw=2*148*NW; int bestR=nny; long best=-1; for(int R=4;R<=nny;++R){ long nb=(nny+R-1)/R; long rounds=((long)nstrips*nb+tw-1)/tw; long cost=rounds*(R+2); if(best<0||cost<best){best=cost;bestR=R;} }
  P.R=bestR; P.nbands=(nny+bestR-1)/bestR; printf("n=%d np=%d lead=%d R=%d nbands=%d units=%d\n",n,np,lead,P.R,P.nbands,nstrips*P.nbands);
  size_t pl=(size_t)np*rows; for(int i=0;i<16;++i){ double* b; CK(cudaMalloc(&b,pl*8)); CK(cudaMemset(b,0,pl*8)); P.a[i]=b+2*(size_t)np+lead; }
  double* out; CK(cudaMalloc(&out,8)); size_t nodes=(size_t)nnx*nny;
  { size_t n2=pl/2; double gb=pl*8.0/1e9; double2* a=(double2*)(P.a[0]-2*(size_t)np-lead); double2* b=(double2*)(P.a[1]-2*(size_t)np-lead);
    timeit("flat set 1 plane",gb,[&]{k_flat_set<<<148*32,256>>>(a,n2,1.0);});
    timeit("flat read 1 plane",gb,[&]{k_flat_read<<<148*8,256>>>(a,out,n2);});
    timeit("flat copy",2*gb,[&]{k_flat_copy<<<148*8,256>>>(a,b,n2);});
    timeit("cudaMemcpy d2d",2*gb,[&]{cudaMemcpyAsync(b,a,pl*8,cudaMemcpyDeviceToDevice);});
  }
  run<10,0,0,0>("10 loads",P,out,nodes);
  run<0,4,0,0>("4 stores",P,out,nodes);
  run<0,1,0,0>("1 store",P,out,nodes);
  run<10,4,0,0>("pass CA: 10 loads + 4 stores",P,out,nodes);
  run<10,4,1,0>("pass CA, one row ahead",P,out,nodes);
  run<10,4,0,1>("pass CA, st.cs",P,out,nodes);
  run<7,1,0,0>("pass B: 7 loads + 1 store",P,out,nodes);
  run<7,1,1,0>("pass B, one row ahead",P,out,nodes);
  run<7,0,1,0>("t recomputed: B' 7 loads",P,out,nodes);
  run<9,4,0,0>("t recomputed: CA' 9 + 4",P,out,nodes);
  run<6,1,1,0>("k_srj: 6 loads + 1 store",P,out,nodes);
  run<1,1,1,0>("marching copy 1 + 1",P,out,nodes);
  return 0;
}
