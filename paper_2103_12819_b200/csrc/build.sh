#!/bin/sh
# Build the C-ABI library in-tree for sm_100a (B200).  Usage: sh build.sh [extra nvcc flags]
set -e
here="$(cd "$(dirname "$0")" && pwd)"
out="$here/../libfdtd_llg.so"
nvcc -O3 -std=c++17 -gencode arch=compute_100a,code=sm_100a -lineinfo \
     -Xcompiler -fPIC -shared "$@" -o "$out" "$here/fdtd_llg.cu"
echo "built $out"
