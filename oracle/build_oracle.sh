#!/bin/sh
# Builds the CPU oracle (test infrastructure): long double parity build and the
# plain-double timed build, both from the one source file.
set -e
cd "$(dirname "$0")"
CFLAGS="-O2 -fno-fast-math -ffp-contract=off -fPIC -shared -fopenmp -Wall -Wextra"
gcc $CFLAGS mopal_oracle.c -o libmopal_oracle.so -lm
gcc $CFLAGS -DORACLE_DOUBLE mopal_oracle.c -o libmopal_oracle_f64.so -lm
