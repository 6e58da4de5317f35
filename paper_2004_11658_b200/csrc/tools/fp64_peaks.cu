// micro-benchmarks: FP64 DFMA / DMMA peaks on B200, layout check of m16n8k16
#include <cstdio>
#include <cstdlib>
#include <cmath>
#include <vector>
#include <cuda_runtime.h>
#define CK(x) do{cudaError_t e=(x); if(e!=cudaSuccess){printf("CUDA error %s at %d\n",cudaGetErrorString(e),__LINE__); exit(1);} }while(0)

__device__ __forceinline__ void mma884(double &c0,double &c1,double a,double b){
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1},{%2},{%3},{%0,%1};\n":"+d"(c0),"+d"(c1):"d"(a),"d"(b));
}
__device__ __forceinline__ void mma1684(double *c,const double *a,double b){
  asm volatile("mma.sync.aligned.m16n8k4.row.col.f64.f64.f64.f64 {%0,%1,%2,%3},{%4,%5},{%6},{%0,%1,%2,%3};\n":"+d"(c[0]),"+d"(c[1]),"+d"(c[2]),"+d"(c[3]):"d"(a[0]),"d"(a[1]),"d"(b));
}
__device__ __forceinline__ void mma1688(double *c,const double *a,const double *b){
  asm volatile("mma.sync.aligned.m16n8k8.row.col.f64.f64.f64.f64 {%0,%1,%2,%3},{%4,%5,%6,%7},{%8,%9},{%0,%1,%2,%3};\n":"+d"(c[0]),"+d"(c[1]),"+d"(c[2]),"+d"(c[3]):"d"(a[0]),"d"(a[1]),"d"(a[2]),"d"(a[3]),"d"(b[0]),"d"(b[1]));
}
__device__ __forceinline__ void mma16816(double *c,const double *a,const double *b){
  asm volatile("mma.sync.aligned.m16n8k16.row.col.f64.f64.f64.f64 {%0,%1,%2,%3},{%4,%5,%6,%7,%8,%9,%10,%11},{%12,%13,%14,%15},{%0,%1,%2,%3};\n":"+d"(c[0]),"+d"(c[1]),"+d"(c[2]),"+d"(c[3]):"d"(a[0]),"d"(a[1]),"d"(a[2]),"d"(a[3]),"d"(a[4]),"d"(a[5]),"d"(a[6]),"d"(a[7]),"d"(b[0]),"d"(b[1]),"d"(b[2]),"d"(b[3]));
}

template<int NCH> __global__ void k_dfma(double *out,int iters,double s){
  double acc[NCH]; 
  #pragma unroll
  for(int i=0;i<NCH;i++) acc[i]=threadIdx.x*1e-3+i;
  double a=s, b=1e-9;
  for(int it=0;it<iters;it++){
    #pragma unroll
    for(int i=0;i<NCH;i++) acc[i]=fma(acc[i],a,b);
  }
  double r=0; 
  #pragma unroll
  for(int i=0;i<NCH;i++) r+=acc[i];
  out[blockIdx.x*blockDim.x+threadIdx.x]=r;
}
template<int NCH> __global__ void k_mma884(double *out,int iters,double s){
  double c0[NCH],c1[NCH];
  #pragma unroll
  for(int i=0;i<NCH;i++){c0[i]=i;c1[i]=-i;}
  double a=s*threadIdx.x,b=1e-9*threadIdx.x;
  for(int it=0;it<iters;it++){
    #pragma unroll
    for(int i=0;i<NCH;i++) mma884(c0[i],c1[i],a,b);
  }
  double r=0;
  #pragma unroll
  for(int i=0;i<NCH;i++) r+=c0[i]+c1[i];
  out[blockIdx.x*blockDim.x+threadIdx.x]=r;
}
template<int NCH,int KK> __global__ void k_mma16(double *out,int iters,double s){
  double c[NCH][4];
  #pragma unroll
  for(int i=0;i<NCH;i++){c[i][0]=i;c[i][1]=-i;c[i][2]=2*i;c[i][3]=3*i;}
  double a[8],b[4];
  #pragma unroll
  for(int i=0;i<8;i++) a[i]=s*(threadIdx.x+i);
  #pragma unroll
  for(int i=0;i<4;i++) b[i]=1e-9*(threadIdx.x+i);
  for(int it=0;it<iters;it++){
    #pragma unroll
    for(int i=0;i<NCH;i++){
      if(KK==4) mma1684(c[i],a,b[0]);
      else if(KK==8) mma1688(c[i],a,b);
      else mma16816(c[i],a,b);
    }
  }
  double r=0;
  #pragma unroll
  for(int i=0;i<NCH;i++) r+=c[i][0]+c[i][1]+c[i][2]+c[i][3];
  out[blockIdx.x*blockDim.x+threadIdx.x]=r;
}
// mixed: NM mma884 + ND dfma per iteration in the same warp
template<int NM,int ND> __global__ void k_mix(double *out,int iters,double s){
  double c0[NM>0?NM:1],c1[NM>0?NM:1],acc[ND>0?ND:1];
  #pragma unroll
  for(int i=0;i<NM;i++){c0[i]=i;c1[i]=-i;}
  #pragma unroll
  for(int i=0;i<ND;i++) acc[i]=i+threadIdx.x;
  double a=s*threadIdx.x,b=1e-9*threadIdx.x;
  for(int it=0;it<iters;it++){
    #pragma unroll
    for(int i=0;i<(NM>ND?NM:ND);i++){
      if(i<NM) mma884(c0[i],c1[i],a,b);
      if(i<ND) acc[i]=fma(acc[i],a,b);
    }
  }
  double r=0;
  #pragma unroll
  for(int i=0;i<NM;i++) r+=c0[i]+c1[i];
  #pragma unroll
  for(int i=0;i<ND;i++) r+=acc[i];
  out[blockIdx.x*blockDim.x+threadIdx.x]=r;
}
// warp-specialised mix: even warps DMMA, odd warps DFMA
__global__ void k_mixw(double *out,int iters,double s,int mma_iters_scale){
  int w=threadIdx.x>>5;
  double r=0;
  if(w&1){
    double acc[16];
    #pragma unroll
    for(int i=0;i<16;i++) acc[i]=i+threadIdx.x;
    for(int it=0;it<iters;it++){
      #pragma unroll
      for(int i=0;i<16;i++) acc[i]=fma(acc[i],s,1e-9);
    }
    #pragma unroll
    for(int i=0;i<16;i++) r+=acc[i];
  } else {
    double c0[16],c1[16];
    #pragma unroll
    for(int i=0;i<16;i++){c0[i]=i;c1[i]=-i;}
    double a=s*threadIdx.x,b=1e-9*threadIdx.x;
    for(int it=0;it<iters*mma_iters_scale/8;it++){
      #pragma unroll
      for(int i=0;i<16;i++) mma884(c0[i],c1[i],a,b);
    }
    #pragma unroll
    for(int i=0;i<16;i++) r+=c0[i]+c1[i];
  }
  out[blockIdx.x*blockDim.x+threadIdx.x]=r;
}

// tanh candidates
__device__ __forceinline__ double tanh_fast(double x){
  // tanh(x) = 1 - 2/(exp(2x)+1), exp via 2^n * p(f)
  double ax=fabs(x);
  ax=fmin(ax,20.0);
  double t=ax*2.8853900817779268; // 2*log2(e)
  double n=rint(t);
  double f=fma(n,-1.0,t)*0.6931471805599453; // f*ln2 in [-.35,.35]
  double p=2.505210838544172e-8; // 1/11!
  p=fma(p,f,2.755731922398589e-7);
  p=fma(p,f,2.7557319223985893e-6);
  p=fma(p,f,2.48015873015873e-5);
  p=fma(p,f,1.984126984126984e-4);
  p=fma(p,f,1.388888888888889e-3);
  p=fma(p,f,8.333333333333333e-3);
  p=fma(p,f,4.1666666666666664e-2);
  p=fma(p,f,1.6666666666666666e-1);
  p=fma(p,f,0.5);
  p=fma(p,f,1.0);
  p=fma(p,f,1.0);
  int ni=(int)n;
  double e=__hiloint2double(__double2hiint(p)+(ni<<20),__double2loint(p));
  double d=e+1.0;
  // reciprocal: fast approx + 2 newton
  double r0=__hiloint2double(0,0);
  asm("rcp.approx.ftz.f64 %0,%1;":"=d"(r0):"d"(d));
  double err=fma(-d,r0,1.0); r0=fma(r0,err,r0);
  err=fma(-d,r0,1.0); r0=fma(r0,err,r0);
  double res=fma(-2.0,r0,1.0);
  return copysign(res,x);
}
template<int MODE> __global__ void k_tanh(double *out,int iters,double s){
  double x[4]; 
  #pragma unroll
  for(int i=0;i<4;i++) x[i]=(threadIdx.x%64)*0.05-1.6+i*0.01+s;
  double r=0;
  for(int it=0;it<iters;it++){
    #pragma unroll
    for(int i=0;i<4;i++){ double y= MODE==0? tanh(x[i]) : tanh_fast(x[i]); r+=y; x[i]=x[i]+y*1e-6; }
  }
  out[blockIdx.x*blockDim.x+threadIdx.x]=r;
}
__global__ void k_tanh_err(double *maxerr){
  double m=0;
  for(int i=threadIdx.x+blockIdx.x*blockDim.x;i<20000000;i+=gridDim.x*blockDim.x){
    double x=-25.0+50.0*(double)i/20000000.0;
    double e=fabs(tanh_fast(x)-tanh(x)); if(e>m)m=e;
    double x2=x*1e-3; e=fabs(tanh_fast(x2)-tanh(x2)); if(e>m)m=e;
  }
  atomicMax((unsigned long long*)maxerr,(unsigned long long)__double_as_longlong(m));
}

// layout check for m16n8k16 and m8n8k4
__global__ void k_layout(const double *A,const double *B,double *C16,double *C8){
  int t=threadIdx.x, g=t/4, q=t%4;
  // m16n8k16: A[16][16] row-major, B[16][8] (k,n)
  double a[8],b[4],c[4]={0,0,0,0};
  for(int i=0;i<8;i++) a[i]=A[(g+8*(i%2))*16 + q+4*(i/2)];
  for(int i=0;i<4;i++) b[i]=B[(q+4*i)*8+g];
  mma16816(c,a,b);
  C16[g*8+2*q]=c[0]; C16[g*8+2*q+1]=c[1]; C16[(g+8)*8+2*q]=c[2]; C16[(g+8)*8+2*q+1]=c[3];
  // m8n8k4: A rows 0..7, k 0..3
  double c0=0,c1=0;
  mma884(c0,c1,A[g*16+q],B[q*8+g]);
  C8[g*8+2*q]=c0; C8[g*8+2*q+1]=c1;
}

template<class F> float timeit(F f,int rep=3){
  cudaEvent_t e0,e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
  f(); CK(cudaDeviceSynchronize());
  float best=1e30f;
  for(int r=0;r<rep;r++){ cudaEventRecord(e0); f(); cudaEventRecord(e1); CK(cudaEventSynchronize(e1)); float ms; cudaEventElapsedTime(&ms,e0,e1); if(ms<best)best=ms; }
  return best;
}

int main(){
  cudaDeviceProp p; CK(cudaGetDeviceProperties(&p,0));
  printf("device %s SMs %d clock %d kHz\n",p.name,p.multiProcessorCount,p.clockRate);
  int nsm=p.multiProcessorCount;
  double *out; CK(cudaMalloc(&out,sizeof(double)*nsm*8*1024));
  int iters=20000;
  for(int bpsm=1;bpsm<=2;bpsm++) for(int th=128;th<=1024;th*=2){
    if(bpsm*th>2048) continue;
    int grid=nsm*bpsm;
    float ms=timeit([&]{k_dfma<16><<<grid,th>>>(out,iters,0.999);});
    printf("DFMA x16 chains grid %d thr %d: %.2f TFLOPS\n",grid,th,2.0*16*iters*(double)grid*th/ms/1e9);
  }
  for(int th=128;th<=1024;th*=2){
    int grid=nsm;
    float ms=timeit([&]{k_mma884<16><<<grid,th>>>(out,iters,0.999);});
    printf("DMMA m8n8k4 x16 grid %d thr %d: %.2f TFLOPS\n",grid,th,2.0*256*16*iters*(double)grid*(th/32)/ms/1e9);
    ms=timeit([&]{k_mma16<8,4><<<grid,th>>>(out,iters,0.999);});
    printf("DMMA m16n8k4 x8 grid %d thr %d: %.2f TFLOPS\n",grid,th,2.0*512*8*iters*(double)grid*(th/32)/ms/1e9);
    ms=timeit([&]{k_mma16<8,8><<<grid,th>>>(out,iters,0.999);});
    printf("DMMA m16n8k8 x8 grid %d thr %d: %.2f TFLOPS\n",grid,th,2.0*1024*8*iters*(double)grid*(th/32)/ms/1e9);
    ms=timeit([&]{k_mma16<8,16><<<grid,th>>>(out,iters/2,0.999);});
    printf("DMMA m16n8k16 x8 grid %d thr %d: %.2f TFLOPS\n",grid,th,2.0*2048*8*(iters/2)*(double)grid*(th/32)/ms/1e9);
  }
  {
    int grid=nsm, th=512;
    float ms=timeit([&]{k_mix<16,16><<<grid,th>>>(out,iters,0.999);});
    printf("MIX same-warp 16 DMMA884 + 16 DFMA: %.3f ms; DMMA-only flops %.2f TF, DFMA flops %.2f TF\n",ms,2.0*256*16*iters*(double)grid*(th/32)/ms/1e9,2.0*16*iters*(double)grid*th/ms/1e9);
    ms=timeit([&]{k_mix<16,4><<<grid,th>>>(out,iters,0.999);});
    printf("MIX same-warp 16 DMMA884 + 4 DFMA: %.3f ms; DMMA flops %.2f TF, DFMA flops %.2f TF\n",ms,2.0*256*16*iters*(double)grid*(th/32)/ms/1e9,2.0*4*iters*(double)grid*th/ms/1e9);
    ms=timeit([&]{k_mix<16,0><<<grid,th>>>(out,iters,0.999);});
    printf("MIX same-warp 16 DMMA884 + 0 DFMA: %.3f ms\n",ms);
    ms=timeit([&]{k_mix<0,16><<<grid,th>>>(out,iters,0.999);});
    printf("MIX same-warp 0 DMMA + 16 DFMA: %.3f ms\n",ms);
    for(int sc=0;sc<=8;sc+=4){
      ms=timeit([&]{k_mixw<<<grid,th>>>(out,iters,0.999,sc);});
      printf("MIXW warp-spec (half warps DFMA %d iters, half DMMA scale %d): %.3f ms\n",iters,sc,ms);
    }
  }
  {
    int grid=nsm*2, th=512; int it2=2000;
    float ms=timeit([&]{k_tanh<0><<<grid,th>>>(out,it2,0.0);});
    printf("tanh libdevice: %.3f ms -> %.2f Gtanh/s\n",ms,4.0*it2*(double)grid*th/ms/1e6);
    ms=timeit([&]{k_tanh<1><<<grid,th>>>(out,it2,0.0);});
    printf("tanh fast: %.3f ms -> %.2f Gtanh/s\n",ms,4.0*it2*(double)grid*th/ms/1e6);
    double *me; CK(cudaMalloc(&me,8)); CK(cudaMemset(me,0,8));
    k_tanh_err<<<nsm*4,256>>>(me); double h; CK(cudaMemcpy(&h,me,8,cudaMemcpyDeviceToHost));
    printf("tanh fast max abs err vs libdevice: %.3e\n",h);
  }
  {
    std::vector<double> A(256),B(128),C16(128),C8(64);
    for(int i=0;i<256;i++)A[i]=sin(i*0.37)+0.1*i; for(int i=0;i<128;i++)B[i]=cos(i*0.11)-0.05*i;
    double *dA,*dB,*dC16,*dC8; CK(cudaMalloc(&dA,2048));CK(cudaMalloc(&dB,1024));CK(cudaMalloc(&dC16,1024));CK(cudaMalloc(&dC8,512));
    CK(cudaMemcpy(dA,A.data(),2048,cudaMemcpyHostToDevice));CK(cudaMemcpy(dB,B.data(),1024,cudaMemcpyHostToDevice));
    k_layout<<<1,32>>>(dA,dB,dC16,dC8); CK(cudaMemcpy(C16.data(),dC16,1024,cudaMemcpyDeviceToHost));CK(cudaMemcpy(C8.data(),dC8,512,cudaMemcpyDeviceToHost));
    double e16=0,e8=0;
    for(int m=0;m<16;m++)for(int n=0;n<8;n++){double r=0;for(int k=0;k<16;k++)r+=A[m*16+k]*B[k*8+n]; e16=fmax(e16,fabs(r-C16[m*8+n]));}
    for(int m=0;m<8;m++)for(int n=0;n<8;n++){double r=0;for(int k=0;k<4;k++)r+=A[m*16+k]*B[k*8+n]; e8=fmax(e8,fabs(r-C8[m*8+n]));}
    printf("layout check: m16n8k16 max err %.3e, m8n8k4 max err %.3e\n",e16,e8);
  }
  return 0;
}
