#!/bin/sh
# Builds the CPU oracle (test infrastructure) twice: double and long double.
# Usage: sh oracle/build.sh   (from anywhere)
set -e
cd "$(dirname "$0")"
SRC="philox_rambo.c lorentz.c colour.c me_eemumu.c me_ggttng.c me_qchannel.c weight.c"
# -O3 -march=native as SURVEY.md §8(d) states for the timed baseline; -ffp-contract=off keeps the arithmetic of every
# formula as written (no fused multiply-adds), so results do not depend on the host CPU
OPT="-O3 -march=native -ffp-contract=off"
gcc $OPT -std=gnu11 -fPIC -shared -fopenmp -Wall -Wno-unknown-pragmas -o liboracle.so $SRC -lm
gcc $OPT -std=gnu11 -fPIC -shared -fopenmp -Wall -Wno-unknown-pragmas -DORACLE_LONG_DOUBLE -o liboracle_ld.so $SRC -lm
