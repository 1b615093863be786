#!/bin/bash
# Builds libmeb_b200.so (sm_100a only) next to this script.  Usage: build.sh [extra nvcc flags]
set -e
cd "$(dirname "$0")"
OUT=libmeb_b200.so
NVCC=${NVCC:-nvcc}
FLAGS="-std=c++17 -O3 -gencode arch=compute_100a,code=sm_100a -lineinfo -Xcompiler -fPIC -Xcompiler -fvisibility=hidden $@"
mkdir -p build
pids=()
for f in csrc/*.cu; do
  o=build/$(basename "${f%.cu}").o
  stale=0
  for h in csrc/*.cuh ../include/meb.h; do [ "$h" -nt "$o" ] && stale=1; done
  if [ ! -f "$o" ] || [ "$f" -nt "$o" ] || [ $stale = 1 ]; then
    $NVCC $FLAGS -c "$f" -o "$o" &
    pids+=($!)
  fi
done
for p in "${pids[@]}"; do wait "$p"; done
$NVCC -shared -gencode arch=compute_100a,code=sm_100a -o $OUT build/*.o -cudart static
echo "built $(pwd)/$OUT"
