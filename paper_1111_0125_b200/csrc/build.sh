#!/bin/sh
# Build libstag.so in-tree for sm_100a.  Usage: sh build.sh [extra nvcc flags]
set -e
here="$(cd "$(dirname "$0")" && pwd)"
nvcc -gencode arch=compute_100a,code=sm_100a -lineinfo -O3 -std=c++17 \
     -Xcompiler -fPIC -shared "$@" \
     -o "$here/../libstag.so.tmp.$$" "$here/stag_lib.cu"
mv "$here/../libstag.so.tmp.$$" "$here/../libstag.so"
