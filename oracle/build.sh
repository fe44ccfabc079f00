#!/bin/sh
# Builds the CPU oracle (test infrastructure) twice: double and long double.
# Usage: sh oracle/build.sh   (from anywhere)
set -e
cd "$(dirname "$0")"
SRC="philox_rambo.c lorentz.c colour.c me_eemumu.c me_ggttng.c"
gcc -O2 -std=gnu11 -fPIC -shared -fopenmp -Wall -Wno-unknown-pragmas -o liboracle.so $SRC -lm
gcc -O2 -std=gnu11 -fPIC -shared -fopenmp -Wall -Wno-unknown-pragmas -DORACLE_LONG_DOUBLE -o liboracle_ld.so $SRC -lm
