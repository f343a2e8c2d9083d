/*
 * simd_loop_probe.c -- what one host core can do with the innermost loop of dedisp_tiled.c.
 *
 * A bound for the tiled CPU baseline (bench.py's cpu_baseline_tiled), not part of it and not part of the
 * product: the loop `S[t] += x[t]` (uint32 or uint16 accumulator, uint8 samples, 4096 samples, unaligned x)
 * run alone on one thread with everything in L1/L2, then with every row fetched from DRAM.  Prints G adds/s.
 *
 *   gcc -std=c99 -O3 -march=native -mprefer-vector-width=512 -fopenmp cpu_tiled/simd_loop_probe.c -o /tmp/p && /tmp/p
 *
 * Results and what they say about the 0.07 T adds/s of the tiled kernel: profiles/r03_cpu_baseline.md.
 */
#include <stdint.h>
#include <stdio.h>
#include <stdlib.h>
#include <time.h>
static double now(){struct timespec t;clock_gettime(CLOCK_MONOTONIC,&t);return t.tv_sec+1e-9*t.tv_nsec;}
int main(){
  int len=4096; size_t N=1<<26; uint8_t*in=malloc(N); for(size_t i=0;i<N;i++)in[i]=i*7;
  uint32_t S[4096]; uint16_t S16[4096];
  for(int t=0;t<len;t++){S[t]=0;S16[t]=0;}
  /* L1-resident x: same 8 rows again and again */
  double t0=now(); long adds=0;
  for(int r=0;r<200000;r++){ const uint8_t*x=in+(r%8)*5000+3+(r%5);
#pragma omp simd
    for(int t=0;t<len;t++)S[t]+=x[t];
    adds+=len;}
  double t1=now(); printf("u32 acc, x in L1/L2: %.1f G adds/s\n",adds/(t1-t0)/1e9);
  t0=now(); adds=0;
  for(int r=0;r<200000;r++){ const uint8_t*x=in+(r%8)*5000+3+(r%5);
#pragma omp simd
    for(int t=0;t<len;t++)S16[t]=(uint16_t)(S16[t]+x[t]);
    adds+=len;}
  t1=now(); printf("u16 acc, x in L1/L2: %.1f G adds/s\n",adds/(t1-t0)/1e9);
  t0=now(); adds=0;
  for(int r=0;r<16000;r++){ const uint8_t*x=in+((size_t)r*262144+3)%(N-8192);
#pragma omp simd
    for(int t=0;t<len;t++)S[t]+=x[t];
    adds+=len;}
  t1=now(); printf("u32 acc, x from DRAM (strided rows): %.1f G adds/s\n",adds/(t1-t0)/1e9);
  uint32_t s=0; for(int t=0;t<len;t++)s+=S[t]+S16[t]; printf("%u\n",s); return 0;}
