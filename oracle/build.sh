#!/bin/sh
# Builds the CPU oracle (test infrastructure) into oracle/libcsph_oracle.so.
# -ffp-contract=off: the CFL time step and the vacuum mask are compared bit for
# bit with the GPU path, so the compiler must not fuse multiplies and adds.
set -e
cd "$(dirname "$0")"
g++ -std=c++17 -O2 -ffp-contract=off -fopenmp -shared -fPIC -o libcsph_oracle.so csph_oracle.cpp
