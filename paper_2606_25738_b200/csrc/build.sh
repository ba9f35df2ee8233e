#!/bin/sh
# Builds libpairhmm_b200.so (sm_100a only) next to the Python binding.  Usage: sh build.sh
set -e
cd "$(dirname "$0")"
OUT=../libpairhmm_b200.so
FLAGS="-gencode arch=compute_100a,code=sm_100a -O3 -lineinfo -std=c++17 -Xcompiler -fPIC -diag-suppress 550"
nvcc $FLAGS -shared -o "$OUT.tmp" phmm_api.cu phmm_short.cu phmm_chain.cu phmm_long.cu phmm_long64.cu phmm_rescue.cu phmm_noalloc.cu phmm_peak.cu phmm_batcher.cpp -lcudart
mv "$OUT.tmp" "$OUT"
echo "built $OUT"
