#!/bin/bash
# The staged GPU session of DESIGN.md section 9 (fault containment): ONE stage per `gpurun` call, in this order,
# and the first non-zero exit stops the session -- the failing kernel, configuration and commit go into
# DESIGN.md section 9 before anything is retried.
#
#   gpurun --timeout 2400 -- 'bash tests/gpu_session.sh memcheck'    # 1. every kernel family at config-0 size under memcheck
#   gpurun --timeout 3600 -- 'bash tests/gpu_session.sh tests'       # 2. pytest -m gpu -x (small -> full size), smoke, bench
#   gpurun --timeout 1800 -- 'bash tests/gpu_session.sh racecheck'   # 3. shared-memory hazards of the FFT kernels (small)
#   gpurun --timeout 2400 -- 'bash tests/gpu_session.sh profile'     # 4. ncu launch list + one --set full capture per top kernel
#
# At most one of ncu / one compute-sanitizer tool per call (B200_PROFILING.md).  Everything is written to gpurun_out/.
set -u
cd "${GRAFT_REPO_ROOT:-$(dirname "$0")/..}" || exit 9
O=gpurun_out
mkdir -p $O
stage=${1:-tests}
SMALL="tests/test_gpu_0_templates.py tests/test_gpu_1_spectrum.py tests/test_gpu_2_correlate.py tests/test_gpu_3_harmsum.py tests/test_gpu_4_host_resample.py tests/test_gpu_5_async_copies.py"
{
nvidia-smi --query-gpu=name,driver_version,clocks.max.sm,memory.total --format=csv
git rev-parse --short HEAD 2>/dev/null
python -c "import __graft_entry__ as g; g.build(); print('build ok')" || exit 8
case $stage in
memcheck)
    # one cudaMalloc per tensor, so that an overrun leaves its allocation instead of landing in the caching allocator's block
    export PYTORCH_NO_CUDA_MEMORY_CACHING=1
    timeout 2000 compute-sanitizer --tool memcheck --error-exitcode 7 python -m pytest $SMALL -x -q -m gpu \
        -k "not 23 and not test_fp32_peak" > $O/memcheck.log 2>&1
    rc=$?; tail -15 $O/memcheck.log; grep -m8 -B2 -A14 "Invalid\|Misaligned\|out of bounds" $O/memcheck.log
    exit $rc ;;
racecheck)
    timeout 1500 compute-sanitizer --tool racecheck --error-exitcode 7 python -m pytest tests/test_gpu_1_spectrum.py \
        tests/test_gpu_2_correlate.py -x -q -m gpu -k "not 20 and not 17" > $O/racecheck.log 2>&1
    rc=$?; tail -15 $O/racecheck.log; grep -m8 -A12 "hazard" $O/racecheck.log
    exit $rc ;;
tests)
    timeout 2400 python -m pytest tests -m gpu -x -q > $O/pytest_gpu.log 2>&1; rc=$?
    tail -15 $O/pytest_gpu.log
    [ $rc -ne 0 ] && { echo "STOP: pytest rc=$rc"; exit 2; }
    timeout 600 python -c "import __graft_entry__ as g; g.smoke()" || { echo "STOP: smoke"; exit 3; }
    timeout 1200 python bench.py --steps 20 --warmup 5 > $O/bench.json 2> $O/bench.err; rc=$?
    cat $O/bench.json; tail -5 $O/bench.err
    [ $rc -ne 0 ] && { echo "STOP: bench rc=$rc"; exit 4; }
    timeout 900 python bench.py --ab --steps 10 > $O/ab.json 2> $O/ab.err; cat $O/ab.json; tail -3 $O/ab.err
    timeout 900 python bench.py --sweep-templates --steps 10 > $O/sweep.json 2> $O/sweep.err; cat $O/sweep.json
    exit 0 ;;
profile)
    CMD="python bench.py --steps 2 --warmup 3 --no-cpu"
    $CMD > $O/plain.log 2>&1 &&
    ncu --metrics gpu__time_duration.sum --clock-control none -c 400 --csv --log-file $O/launches.csv $CMD > $O/ncu_list.log 2>&1 &&
    ncu --set full --clock-control none --import-source on -k regex:k_correlate_2048 -s 3 -c 1 -o $O/prof_correlate $CMD > $O/ncu_corr.log 2>&1 &&
    ncu --set full --clock-control none --import-source on -k regex:k_harmsum -s 3 -c 1 -o $O/prof_harmsum $CMD > $O/ncu_hs.log 2>&1 &&
    ncu --set full --clock-control none --import-source on -k regex:k_spec_ -s 12 -c 4 -o $O/prof_spectrum $CMD > $O/ncu_spec.log 2>&1
    rc=$?; tail -5 $O/plain.log; ls -la $O
    exit $rc ;;
*) echo "unknown stage $stage"; exit 9 ;;
esac
} 2>&1 | tee $O/session_$stage.log
exit ${PIPESTATUS[0]}
