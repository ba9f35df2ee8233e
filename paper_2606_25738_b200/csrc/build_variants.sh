#!/bin/sh
# Compile-time variants of libpairhmm_b200.so for the columns-per-thread x occupancy sweep (Fig.5;
# SURVEY.md section 8(f) item 1).  Usage: sh build_variants.sh OUTDIR
#   fp32 short kernel: SHORT_NV_ = 8 | 16 columns per virtual lane (16 | 32 per thread), SHORT_MIN_CTAS = resident CTAs per SM
#   fp64 sub-warp kernels: RESCUE_NV_ = 16 | 32 columns per lane, RESCUE_MIN_CTAS = resident CTAs per SM
# The variant in use is chosen with the PHMM_LIB environment variable (binding.py); results: profiles/r2_gn_sweep.md.
set -e
cd "$(dirname "$0")"
OUT=${1:?usage: sh build_variants.sh OUTDIR}
mkdir -p "$OUT"
FLAGS="-gencode arch=compute_100a,code=sm_100a -O3 -lineinfo -std=c++17 -Xcompiler -fPIC -diag-suppress 550"
SRC="phmm_api.cu phmm_short.cu phmm_chain.cu phmm_long.cu phmm_long64.cu phmm_rescue.cu phmm_noalloc.cu phmm_peak.cu phmm_batcher.cpp"
for v in "nv16_c3:-DSHORT_NV_=16 -DSHORT_MIN_CTAS=3" "nv16_c2:-DSHORT_NV_=16 -DSHORT_MIN_CTAS=2" "nv16_c4:-DSHORT_NV_=16 -DSHORT_MIN_CTAS=4" \
         "nv8_c3:-DSHORT_NV_=8 -DSHORT_MIN_CTAS=3" "nv8_c4:-DSHORT_NV_=8 -DSHORT_MIN_CTAS=4" "nv8_c5:-DSHORT_NV_=8 -DSHORT_MIN_CTAS=5" \
         "dnv32_c2:-DRESCUE_NV_=32 -DRESCUE_MIN_CTAS=2" "dnv16_c2:-DRESCUE_NV_=16 -DRESCUE_MIN_CTAS=2" "dnv16_c3:-DRESCUE_NV_=16 -DRESCUE_MIN_CTAS=3" \
         "dnv16_c4:-DRESCUE_NV_=16 -DRESCUE_MIN_CTAS=4"; do
    name=${v%%:*}; defs=${v#*:}
    nvcc $FLAGS $defs -shared -o "$OUT/libpairhmm_$name.so" $SRC -lcudart &
done
wait
ls -1 "$OUT"
