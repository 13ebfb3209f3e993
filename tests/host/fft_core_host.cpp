// Host check of the device FFT core (csrc/fft_core.cuh is plain C++ when compiled without nvcc): the 32-point
// register DFT fft32 against a naive fp64 DFT, and the index maps of the register-resident path of mk_fft_fast.cu
// (four-step 1024 = 32 x 32 with one padded transposition; radix-2 split for nt = 4096) replayed lane by lane.
// Built and run by tests/test_fft_core_host.py; exit code 0 = all errors below the thresholds.
#include <cstdio>
#include <complex>
#include <vector>
#include <cmath>
#include <cstdlib>
#include "fft_core.cuh"
using namespace mkfft;
typedef std::complex<double> cd;
static const int SUB = 32*33;
static std::vector<float2> tw1k(1024);
template<bool INV> void warp_fft1024(float2 a[32][32] /*[lane][reg]*/, float2* scratch) {
  for (int t=0;t<32;++t){ fft32<INV>(a[t]); for(int k1=1;k1<32;++k1){ float2 w=tw1k[k1*32+t]; a[t][k1]= INV? cmulc(a[t][k1],w):cmul(a[t][k1],w);} }
  for (int t=0;t<32;++t) for(int k1=0;k1<32;++k1) scratch[k1*33+t]=a[t][k1];
  for (int t=0;t<32;++t){ for(int n2=0;n2<32;++n2) a[t][n2]=scratch[t*33+n2]; fft32<INV>(a[t]); }
}
int main(){
  int bad=0;
  const double PI=3.14159265358979323846;
  for(int k1=0;k1<32;++k1)for(int t=0;t<32;++t){double a=-2*PI*k1*t/1024.0; tw1k[k1*32+t]=make_float2((float)cos(a),(float)sin(a));}
  // fft32 test
  { float2 a[32]; cd x[32]; for(int i=0;i<32;++i){x[i]=cd(drand48()-.5,drand48()-.5); a[i]=make_float2((float)x[i].real(),(float)x[i].imag());}
    float2 b[32]; for(int i=0;i<32;++i)b[i]=a[i];
    fft32<false>(a); fft32<true>(b); double e=0,e2=0; for(int k=0;k<32;++k){cd s=0,s2=0; for(int n=0;n<32;++n){s+=x[n]*std::polar(1.0,-2*PI*k*n/32); s2+=x[n]*std::polar(1.0,2*PI*k*n/32);} e=fmax(e,abs(s-cd(a[k].x,a[k].y))); e2=fmax(e2,abs(s2-cd(b[k].x,b[k].y)));}
    printf("fft32 fwd err %.2e inv err %.2e\n",e,e2); if(!(e<3e-6&&e2<3e-6)) bad=1;}
  for (int HF=1; HF<=2; ++HF){
    const int M=1024*HF, nt=2*M;
    std::vector<float2> tw(nt); for(int k=0;k<nt;++k){double a=-2*PI*k/nt; tw[k]=make_float2((float)cos(a),(float)sin(a));}
    std::vector<cd> Z(M); for(auto&z:Z) z=cd(drand48()-.5,drand48()-.5);
    std::vector<float2> buf(HF*SUB+2);
    auto zaddr=[&](int k){return (k>>10)*SUB+((k&1023)>>5)*33+(k&31);};
    for(int k=0;k<M;++k) buf[zaddr(k)]=make_float2((float)Z[k].real(),(float)Z[k].imag());
    // inverse
    static float2 a[2][32][32];
    for(int hf=0;hf<HF;++hf)for(int t=0;t<32;++t)for(int n1=0;n1<32;++n1){
      if(HF==1) a[hf][t][n1]=buf[n1*33+t];
      else { float2 z0=buf[n1*33+t], z1=buf[SUB+n1*33+t];
        if(hf==0) a[hf][t][n1]=cadd(z0,z1); else a[hf][t][n1]=cmulc(csub(z0,z1), tw[(32*n1+t)*(nt/2048)]); } }
    for(int hf=0;hf<HF;++hf) warp_fft1024<true>(a[hf], buf.data()+hf*SUB);
    // check: a[hf][t][q] = out[HF*(t+32q)+hf]
    double e=0; std::vector<cd> out(M);
    for(int n=0;n<M;++n){cd s=0; for(int k=0;k<M;++k) s+=Z[k]*std::polar(1.0,2*PI*(double)k*n/M); out[n]=s;}
    for(int hf=0;hf<HF;++hf)for(int t=0;t<32;++t)for(int q=0;q<32;++q){int m=HF*(t+32*q)+hf; e=fmax(e,abs(out[m]-cd(a[hf][t][q].x,a[hf][t][q].y)));}
    printf("HF=%d inverse max err %.2e (values ~%g)\n",HF,e,sqrt((double)M)*0.4); if(!(e<5e-5)) bad=1;
    // forward of these registers; expect M*Z
    for(int hf=0;hf<HF;++hf){ warp_fft1024<false>(a[hf], buf.data()+hf*SUB);
      for(int t=0;t<32;++t)for(int k2=0;k2<32;++k2){ float2 v=a[hf][t][k2]; if(HF==2&&hf==1) v=cmul(v,tw[(t+32*k2)*(nt/2048)]); buf[hf*SUB+k2*33+t]=v; } }
    double e2=0;
    for(int k=0;k<M;++k){ cd z; if(HF==1){float2 v=buf[zaddr(k)]; z=cd(v.x,v.y);} else {int kp=k&1023; int ad=(kp>>5)*33+(kp&31); float2 E=buf[ad],O=buf[SUB+ad]; float2 v= k<1024? cadd(E,O):csub(E,O); z=cd(v.x,v.y);} 
      e2=fmax(e2,abs(z/(double)M-Z[k])); }
    printf("HF=%d forward(inverse) roundtrip max err %.2e\n",HF,e2); if(!(e2<2e-6)) bad=1;
  }
  return bad;
}
