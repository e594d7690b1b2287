#!/bin/bash
# The GPU gate of DESIGN.md 9a, step 1, as one command for the first GPU call on a new build (run from the repository root):
#
#     bash tests/gpu_gate.sh [output directory, default gpurun_out]
#
# Order: the index-checked build (-DHOUGH_BOUNDS: a failed check is counted and the access skipped, nothing traps) on the small
# gate cases, then on every GPU test; only then the product build, small cases first.  Stops at the first failing step, so that a
# wrong build never reaches a full-size launch.  compute-sanitizer (memcheck, then racecheck: one tool per GPU call) and bench.py
# come after this script has passed; DESIGN.md 9a has the commands.
set -u
out=${1:-gpurun_out}
mkdir -p "$out"
step() {
    local name=$1; shift
    echo "== $name: $*"
    if ! timeout 3000 "$@" > "$out/gate_$name.log" 2>&1; then
        echo "== $name FAILED (see $out/gate_$name.log); the later steps were not run"
        tail -25 "$out/gate_$name.log"
        exit 1
    fi
    tail -1 "$out/gate_$name.log"
}
step build_bounds   python -m paper_2511_02742_b200.build --variant=bounds
step build_product  python -m paper_2511_02742_b200.build
step bounds_small   python -m pytest tests -m gpu --gate --hough-variant=bounds -x -q
step bounds_all     python -m pytest tests -m gpu --hough-variant=bounds -x -q
step product_small  python -m pytest tests -m gpu --gate -x -q
step product_all    python -m pytest tests -m gpu -x -q
echo "== gate passed"
