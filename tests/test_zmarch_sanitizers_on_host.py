"""The sweep kernel on the host execution model (tests/host_emul/, see tests/test_zmarch_on_host.py) under the compiler's
sanitizers.  No GPU; it is what can be done here of the compute-sanitizer record the kernel should have.

* ThreadSanitizer = a race check of the CTA-level shared-memory protocol: every CUDA thread is an OS thread, __syncthreads and
  the warp shuffles are pthread barriers, so a shared-memory (or global-memory) store and a load of the same bytes by two
  threads with no barrier between them is a data race the tool reports, whether or not it changed the spins of this run.
  A seeded fault (the barrier that ends a step removed) must be reported.  What it cannot see: the model's mbarriers and its
  cluster barrier are mutexes, which order MORE than the hardware's do, so a missing mbarrier wait may go unreported here —
  that kind of fault is what the early / late landing modes of tests/test_zmarch_on_host.py detect by wrong bits.
* AddressSanitizer = memcheck: spins, J / H, E / m and the CTA's shared memory are heap blocks of exactly their stated sizes.

The race check runs every lattice size of the kernel (the L = 64 thread-block cluster included) and the smallest and the
largest group size, the memory check L = 16 and the cluster kernel."""
import shutil
import subprocess
from concurrent.futures import ThreadPoolExecutor
from pathlib import Path

import pytest

import oracle

ROOT = Path(__file__).resolve().parent.parent
CSRC = ROOT / "paper_1204_6192_b200" / "csrc"
HERE = Path(__file__).resolve().parent
SOURCES = [CSRC / "hsg_zmarch.cuh", CSRC / "hsg_zmarch_launch.h", CSRC / "hsg_layout.cuh", CSRC / "hsg_math.cuh",
           HERE / "host_math" / "cuda_runtime.h", HERE / "host_math" / "hsg_prim.cuh", HERE / "host_emul" / "emu.h",
           HERE / "host_emul" / "hsg_zmarch_ptx.cuh", HERE / "host_emul" / "zmarch_driver.cpp", HERE / "host_emul" / "sanitizer_main.cpp"]
SIZES = (8, 16, 32, 64)
ASAN_SIZES = (16, 64)          # the memory check on one single-CTA size and on the cluster kernel (the suite's time)
ENV = {"TSAN_OPTIONS": "halt_on_error=0 exitcode=66", "ASAN_OPTIONS": "detect_leaks=0 exitcode=66", "PATH": "/usr/bin:/bin"}


def _remove_step_barrier(s):
    return s.replace("void step_end() {\n  cta_sync();", "void step_end() {\n", 1)


def _compile(d: Path, L, tool, edit=None):
    for p in SOURCES:
        shutil.copy(p, d / p.name)
    if edit is not None:
        k = d / "hsg_zmarch.cuh"
        text = k.read_text()
        new = edit(text)
        assert new != text, "the edit did not change the kernel source"
        k.write_text(new)
    flags = ["-O1", "-std=c++17", "-ffp-contract=off", "-fno-fast-math", "-Wno-unknown-pragmas", "-pthread",
             f"-fsanitize={tool}", "-fno-omit-frame-pointer", "-I", str(d)]
    if oracle._cpu_has_fma():
        flags.append("-mfma")
    out = d / f"{tool}_l{L}"
    r = subprocess.run(["g++", *flags, f"-DEMU_L={L}", str(d / "zmarch_driver.cpp"), str(d / "sanitizer_main.cpp"), "-o", str(out)],
                       capture_output=True, text=True)
    return out if r.returncode == 0 else None


@pytest.fixture(scope="module")
def programs(tmp_path_factory):
    """(tool, L) -> executable, plus ("thread", "fault") = the kernel without its step barrier at L = 16; None where the
    sanitizer's runtime is not installed."""
    jobs = [("thread", L, None) for L in SIZES] + [("address", L, None) for L in ASAN_SIZES] + [("thread", "fault", _remove_step_barrier)]

    base = tmp_path_factory.mktemp("zmarch_sanitizers")

    def one(job):
        tool, L, edit = job
        d = base / f"{tool}_{L}"
        d.mkdir()
        return (tool, L), _compile(d, 16 if L == "fault" else L, tool, edit)
    with ThreadPoolExecutor(max_workers=8) as ex:
        return dict(ex.map(one, jobs))


def _run(prog, *args, env=ENV):
    if prog is None:
        pytest.skip("this sanitizer's runtime library is not installed")
    r = subprocess.run([str(prog), *map(str, args)], capture_output=True, text=True, env=env, timeout=600)
    if "unexpected memory mapping" in r.stderr or "Shadow memory range interleaves" in r.stderr:
        pytest.skip("the sanitizer cannot map its shadow memory in this container")
    return r


# (L, G, D, O, T, n_or, n_hb): several warps per CTA wherever the size allows, several samples, both kinds of sweep
# (several sweeps per launch at the small sizes: the rings run on across the sweeps of a call)
CASES = [(8, 8, 1, 2, 4, 3, 2), (8, 1, 1, 1, 3, 1, 1), (16, 8, 1, 2, 4, 2, 1), (16, 4, 1, 2, 2, 1, 1),
         (32, 2, 1, 2, 1, 2, 1), (64, 1, 1, 1, 1, 1, 1)]
RUNS = [("thread", c) for c in CASES] + [("address", c) for c in CASES if c[0] in ASAN_SIZES and c[1] != 4]


@pytest.mark.parametrize("tool,case", RUNS, ids=[f"L{c[0]}-G{c[1]}-{tool}" for tool, c in RUNS])
def test_sweep_kernel_on_the_host_model_is_clean_under_the_sanitizer(programs, tool, case):
    L, G, D, O, T, n_or, n_hb = case
    # landing modes: both for the race check of the small sizes; one where a run takes ten seconds and more (copies landing at
    # issue, by the issuing thread, is the mode that exposes a slot refilled too early); the mode moves no address, so one
    # is enough for the memory check
    for mode in ((0, 1) if tool == "thread" and L <= 16 else (0,)):
        r = _run(programs[(tool, L)], G, D, O, T, n_or, n_hb, mode)
        assert r.returncode == 0 and "Sanitizer" not in r.stderr, r.stderr[-4000:]
        assert "rc=0" in r.stdout


def test_thread_sanitizer_reports_a_missing_step_barrier(programs):
    """Sensitivity of the race check: without the __syncthreads that ends a step, a ring slot is refilled while another warp
    still reads it (L = 16, G = 8: several warps per CTA)."""
    # (stop at the first report: a kernel without its barrier need not terminate)
    r = _run(programs[("thread", "fault")], 8, 1, 2, 4, 1, 1, 0, env=dict(ENV, TSAN_OPTIONS="halt_on_error=1 exitcode=66"))
    assert r.returncode == 66 and "ThreadSanitizer: data race" in r.stderr
