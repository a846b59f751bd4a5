"""The boundary from plain C, and the host runtime under sanitizers (no GPU).

(1) include/hadpsgd.h must be a C header: tests/abi_host_check.c is compiled as C99 with
    -Wall -Werror -pedantic, linked against libhadpsgd.so, and run.
(2) compute-sanitizer is closed on the GPU pool, so the host half of the product (allocator,
    scheduler, schedule helpers -- pure C++) is at least run under ASan + UBSan: the same C client is
    built together with those sources and -fsanitize=address,undefined.
(3) hypothesis: random segment tables keep the allocator's invariants."""
import os
import subprocess

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
INC = os.path.join(ROOT, "include")
CSRC = os.path.join(ROOT, "paper_1907_05701_b200", "csrc")
CLIENT = os.path.join(ROOT, "tests", "abi_host_check.c")


@pytest.fixture(scope="module")
def H():
    from paper_1907_05701_b200 import build as b
    b.build()
    import paper_1907_05701_b200 as m
    return m


def test_header_is_c_and_client_runs_against_the_shared_library(H, tmp_path):
    exe = tmp_path / "abi_host_check"
    libdir = os.path.join(ROOT, "paper_1907_05701_b200")
    subprocess.run(["gcc", "-std=c99", "-Wall", "-Wextra", "-Werror", "-pedantic", "-I", INC, CLIENT, "-o", str(exe),
                    "-L", libdir, "-lhadpsgd", f"-Wl,-rpath,{libdir}"], check=True)
    r = subprocess.run([str(exe)], capture_output=True, text=True, timeout=120)
    assert r.returncode == 0 and r.stdout.strip() == "ok", r.stderr


def test_host_runtime_under_asan_ubsan(tmp_path):
    obj = tmp_path / "client.o"
    exe = tmp_path / "abi_host_check_san"
    san = ["-fsanitize=address,undefined", "-fno-sanitize-recover=all", "-fno-omit-frame-pointer", "-g", "-O1"]
    subprocess.run(["gcc", "-std=c99", "-I", INC, *san, "-c", CLIENT, "-o", str(obj)], check=True)
    # hadpsgd_error_string lives in the CUDA translation unit; give the sanitizer build a stand-in
    stub = tmp_path / "stub.cpp"
    stub.write_text('extern "C" const char* hadpsgd_error_string(int c) { return c == 0 ? "ok" : "error"; }\n')
    subprocess.run(["g++", "-std=c++17", "-I", INC, *san, str(obj), str(stub), os.path.join(CSRC, "allocator.cpp"),
                    os.path.join(CSRC, "scheduler.cpp"), os.path.join(CSRC, "schedule.cpp"), "-o", str(exe)], check=True)
    env = dict(os.environ, ASAN_OPTIONS="detect_leaks=1:abort_on_error=0", UBSAN_OPTIONS="print_stacktrace=1")
    r = subprocess.run([str(exe)], capture_output=True, text=True, timeout=300, env=env)
    assert r.returncode == 0 and r.stdout.strip() == "ok", r.stderr[-2000:]


def test_allocator_invariants_on_random_tables(H):
    from hypothesis import given, settings, strategies as st

    @settings(max_examples=150, deadline=None)
    @given(st.lists(st.integers(1, 5000), min_size=1, max_size=40), st.integers(1, 16), st.integers(1, 9),
           st.sampled_from([H.F32, H.BF16]), st.sampled_from([H.F32, H.BF16]))
    def check(seg, S, G, gd, wd):
        lay = H.hadpsgd_layout(S, G, seg, gd, wd)
        off, P = lay["seg_offset"], lay["P_padded"]
        ends = [o + n for o, n in zip(off, seg)]
        assert off[0] == 0 and all(o % 64 == 0 for o in off) and P % 64 == 0
        assert all(e <= o2 for e, o2 in zip(ends, off[1:])) and ends[-1] <= P          # disjoint, inside
        assert all(o2 - e < 64 for e, o2 in zip(ends, off[1:])) and P - ends[-1] < 64  # minimal padding
        eb = 2 if gd == H.BF16 else 4
        assert lay["w_off"] == 0 and lay["v_off"] >= S * P * 4 and lay["g_off"] >= lay["v_off"] + S * P * 4
        need = H.hadpsgd_required_bytes(S, G, seg, gd, wd)
        assert need >= lay["g_off"] + S * G * P * eb + (S * P * 2 if wd == H.BF16 else 0)
        assert all(lay[k] % 256 == 0 for k in ("w_off", "v_off", "g_off", "wb_off"))
        if wd == H.BF16:
            assert lay["wb_off"] >= lay["g_off"] + S * G * P * eb

    check()
