/* latency.c — synchronous-call latency of mf_nll_grad / mf_nll_grad_hess from C, by kernel launch and through the resident
 * evaluation kernel (mf_model_serve), and a full mf_fit.  Build (from the repo root):
 *   gcc -O2 -I include -o latency paper_2505_12414_b200/examples/latency.c -L paper_2505_12414_b200/lib -lmorefit_b200 \
 *       -Wl,-rpath,$PWD/paper_2505_12414_b200/lib -lm
 * Usage: ./latency [n_events]   (events are uniform in the mass range: a timing input, not a physics sample) */
#include <stdio.h>
#include <stdlib.h>
#include <time.h>
#include <math.h>
#include "morefit_b200.h"
static double now(void){struct timespec t;clock_gettime(CLOCK_MONOTONIC,&t);return t.tv_sec+1e-9*t.tv_nsec;}
int main(int argc,char**argv){
  int64_t n = argc>1?atoll(argv[1]):10000;
  mf_ctx*ctx; if(mf_ctx_create(0,NULL,&ctx)) return 1;
  double*m=malloc(8*n); unsigned s=1; for(int64_t i=0;i<n;++i){s=s*1664525u+1013904223u; m[i]=5.0+0.6*(s>>8)/16777216.0;}
  const double*cols[1]={m}; double lo=5.0,hi=5.6; mf_dataset*ds; if(mf_dataset_upload(ctx,1,n,1,cols,MF_HOST,&lo,&hi,&ds)) return 2;
  mf_model*md; if(mf_model_create(ctx,MF_MASS_GAUSS_EXP,ds,&md)) return 3;
  double lam[4]={0.5,5.27,0.03,-1.0},nll,g[4],h[16];
  for(int served=0;served<2;++served){
    mf_model_serve(md,served);
    for(int i=0;i<200;++i) mf_nll_grad(md,lam,&nll,g);
    double t=now(); for(int i=0;i<5000;++i) mf_nll_grad(md,lam,&nll,g); double dt=(now()-t)/5000*1e6;
    double t2=now(); for(int i=0;i<5000;++i) mf_nll_grad_hess(md,lam,&nll,g,h); double dt2=(now()-t2)/5000*1e6;
    printf("n=%lld served=%d nll=%.12g  grad call %.2f us  hess call %.2f us\n",(long long)n,served,nll,dt,dt2);
  }
  mf_model_serve(md,0);
  { /* throughput of evaluations issued one at a time WITHOUT waiting (mf_nll_grad_points with one point = mf_nll_grad_async:
       one launch each, pipelined on the GPU) and of 8-point calls (one launch per call), results on the device */
    double *lam8=malloc(8*4*8), nb; int64_t nbad; double nll8[8], g8[32];
    for(int p=0;p<8;++p){lam8[4*p]=0.5+0.001*p; lam8[4*p+1]=5.27; lam8[4*p+2]=0.03; lam8[4*p+3]=-1.0;}
    /* device output rows come from a sweep's scratch: use mf_nll_grad_sweep once to size it, then the async entry points need a
       device pointer, which C callers get from their own cudaMalloc; here the sweep (host results) is timed instead */
    for(int i=0;i<50;++i) mf_nll_grad_sweep(md,8,lam8,nll8,g8,&nbad);
    double t=now(); for(int i=0;i<2000;++i) mf_nll_grad_sweep(md,8,lam8,nll8,g8,&nbad); double dt=(now()-t)/2000*1e6;
    printf("n=%lld sweep of 8 points (one call, host results): %.2f us per call = %.2f us per evaluation\n",(long long)n,dt,dt/8); (void)nb;
    free(lam8);
  }
  mf_fit_result r; double t=now(); mf_fit(md,lam,NULL,NULL,&r); printf("fit %.1f us calls %d conv %d\n",(now()-t)*1e6,r.n_calls,r.converged);
  t=now(); mf_fit(md,lam,NULL,NULL,&r); printf("fit %.1f us calls %d conv %d\n",(now()-t)*1e6,r.n_calls,r.converged);
  mf_model_destroy(md); mf_dataset_destroy(ds); mf_ctx_destroy(ctx); return 0;}
