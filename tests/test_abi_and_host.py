"""CPU-side checks (no GPU): the C-ABI library loads and exports every symbol include/dia.h declares, argument
errors are caught on the host, the struct layouts of the binding match the header, and the epoch sharding used
by the multi-GPU mode works under a 2-rank gloo group."""
import ctypes as C
import os
import re
import socket
import subprocess
import sys
import textwrap

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared_functions(header):
    src = open(header).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(dia_[a-z0-9_]+)\s*\(", src)))


def test_library_exports_every_declared_symbol():
    import paper_2104_13715_b200 as dia
    lib = dia.load_library()
    declared = _declared_functions(os.path.join(ROOT, "include", "dia.h"))
    assert set(declared) == set(dia.EXPORTED_SYMBOLS), declared
    for name in declared:
        assert getattr(lib, name) is not None
    # the oracle library is a separate binary with its own prefix and header
    import oracle.build
    ref = C.CDLL(oracle.build.build())
    for name in _declared_functions(os.path.join(ROOT, "oracle", "dia_ref.h")):
        assert name.startswith("dia_ref_") and getattr(ref, name) is not None


def test_no_shared_code_between_oracle_and_cuda_path():
    """The two implementations share no source, header or helper, and neither imports the other."""
    for dirpath, _, files in os.walk(os.path.join(ROOT, "paper_2104_13715_b200")):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert "oracle" not in text and "dia_ref" not in text, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c", ".h")):
            text = open(os.path.join(ROOT, "oracle", f)).read()
            assert not re.search(r'#include\s+"[^"]*dia\.h"', text.replace("dia_ref.h", "")) and "libdia_b200" not in text, f
            assert not re.search(r"^\s*(from|import)\s+paper_2104_13715_b200", text, flags=re.M), f
    for f in os.listdir(os.path.join(ROOT, "workloads")):
        if f.endswith(".py"):
            text = open(os.path.join(ROOT, "workloads", f)).read()
            assert not re.search(r"^\s*(from|import)\s+(oracle|paper_2104_13715_b200)", text, flags=re.M), f


def test_default_fit_opts_match_header_and_oracle():
    import oracle
    import paper_2104_13715_b200 as dia
    og, oo = dia.FitOpts.default(), oracle.RefFitOpts.default()
    assert og.lr_kernel == pytest.approx(1e-3) and og.lr_b0 == 10.0
    assert og.tol_switch == 1e-6 and og.tol_change_rel == 1e-8 and og.tol_grad_abs == 1e-7
    assert og.lbfgs_lr == 1.0 and og.lbfgs_history == 100 and og.lbfgs_backtrack == 0
    for name, _ in dia.FitOpts._fields_:
        assert float(getattr(og, name)) == pytest.approx(float(getattr(oo, name)), rel=1e-7), name


def test_binding_struct_layouts_match_header(tmp_path):
    """sizeof / offsetof of the ctypes mirrors against the header compiled by gcc (plain C, no CUDA)."""
    import paper_2104_13715_b200 as dia
    from paper_2104_13715_b200.binding import _Config
    src = tmp_path / "layout.c"
    src.write_text('#include <stdio.h>\n#include <stddef.h>\n#include "dia.h"\nint main(void) {\n'
                   'printf("%zu %zu %zu %zu %zu %zu %zu\\n", sizeof(dia_config), sizeof(dia_fit_opts), '
                   'sizeof(dia_fit_result), offsetof(dia_config, d_flat), offsetof(dia_fit_opts, tol_change_rel), '
                   'offsetof(dia_fit_opts, force_adam_iters), offsetof(dia_fit_result, n_adam));\nreturn 0; }\n')
    exe = tmp_path / "layout"
    subprocess.run(["gcc", "-std=c99", "-I", os.path.join(ROOT, "include"), "-o", str(exe), str(src)], check=True)
    got = [int(x) for x in subprocess.run([str(exe)], capture_output=True, text=True, check=True).stdout.split()]
    want = [C.sizeof(_Config), C.sizeof(dia.FitOpts), C.sizeof(dia.FitResult), _Config.d_flat.offset,
            dia.FitOpts.tol_change_rel.offset, dia.FitOpts.force_adam_iters.offset, dia.FitResult.n_adam.offset]
    assert got == want


def test_status_strings_and_host_side_argument_errors():
    """Argument errors are detected on the host before any launch; without a CUDA device dia_create fails
    with DIA_ERR_CUDA (there is no CPU fallback)."""
    import torch
    import paper_2104_13715_b200 as dia
    lib = dia.load_library()
    assert lib.dia_status_string(0) == b"ok" and lib.dia_status_string(-4) == b"unsupported configuration"
    assert lib.dia_destroy(None) == -1
    out = C.c_void_p()
    assert lib.dia_create(None, None, C.byref(out)) == -1
    assert b"null" in lib.dia_last_error(None)
    with pytest.raises(dia.DiaError):
        dia.dia_create(8, 8, 3, torch.zeros((8, 8)))                            # host tensor is refused by the binding
    if not torch.cuda.is_available():
        from paper_2104_13715_b200.binding import _Config
        cfg = _Config(16, 16, 3, 1, 0, 1.345, 0, 5.0, 1.0, None, None)
        buf = (C.c_float * 256)()
        rc = lib.dia_create(C.byref(cfg), C.cast(buf, C.c_void_p), C.byref(out))
        assert rc == -2 and out.value is None                                   # DIA_ERR_CUDA, no fallback
        cfg.m = 4
        assert lib.dia_create(C.byref(cfg), C.cast(buf, C.c_void_p), C.byref(out)) == -1
        cfg.m, cfg.n_rows, cfg.n_cols = 49, 64, 64
        assert lib.dia_create(C.byref(cfg), C.cast(buf, C.c_void_p), C.byref(out)) == -4
        peak = C.c_double()
        assert lib.dia_measure_fp32_peak(None, C.byref(peak)) == -2


def test_epoch_shard_partition():
    from paper_2104_13715_b200.sharding import epoch_shard
    for E in (0, 1, 7, 16, 33):
        for world in (1, 2, 3, 8):
            spans = [epoch_shard(E, world, r) for r in range(world)]
            assert spans[0][0] == 0 and spans[-1][1] == E
            assert all(spans[r][1] == spans[r + 1][0] for r in range(world - 1))
            sizes = [b - a for a, b in spans]
            assert max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        epoch_shard(4, 2, 2)


_WORKER = textwrap.dedent("""
    import os, sys
    sys.path.insert(0, {root!r})
    import torch, torch.distributed as dist
    from paper_2104_13715_b200.sharding import epoch_shard, gather_epochs, max_over_ranks
    dist.init_process_group("gloo")
    rank, world = dist.get_rank(), dist.get_world_size()
    E, npar = 5, 4
    a, b = epoch_shard(E, world, rank)
    # each rank "fits" its own epochs: row e holds e in every column
    local = torch.arange(a, b, dtype=torch.float32)[:, None].repeat(1, npar)
    full = gather_epochs(local, E)
    assert full.shape == (E, npar) and torch.equal(full[:, 0], torch.arange(E, dtype=torch.float32)), full
    t = max_over_ranks(10.0 + rank)
    assert t == 10.0 + world - 1
    dist.destroy_process_group()
    print("rank%d-ok" % rank, flush=True)
    sys.stdout.flush()
""")


def test_epoch_sharding_two_ranks_gloo(tmp_path):
    """N > 1 path on CPU: 2 processes, gloo backend, epochs sharded with no data-path collective; only the
    fitted parameters are gathered and the device time is max-reduced."""
    script = tmp_path / "worker.py"
    script.write_text(_WORKER.format(root=ROOT))
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node=2",
           "--master-addr", "127.0.0.1", "--master-port", str(port), str(script)]
    out = subprocess.run(cmd, capture_output=True, text=True, timeout=240)
    assert out.returncode == 0, out.stdout + out.stderr
    assert "rank0-ok" in out.stdout and "rank1-ok" in out.stdout, out.stdout


_BAND_WORKER = textwrap.dedent("""
    import os, sys
    sys.path.insert(0, {root!r})
    import numpy as np, torch, torch.distributed as dist
    import oracle
    from workloads import make_workload
    from paper_2104_13715_b200.sharding import row_band, sum_over_ranks_in_order
    dist.init_process_group("gloo")
    rank, world = dist.get_rank(), dist.get_world_size()
    w = make_workload(0, n=61, m=5)                      # 57 valid rows: bands of 29 and 28
    th = w.theta_true[0].astype(np.float32)
    v0, v1, i0, i1 = row_band(w.n, w.m, world, rank)
    assert i1 - i0 == (v1 - v0) + w.m - 1
    cfg = oracle.RefConfig(i1 - i0, w.n, w.m, sigma0=w.sigma0, gain=w.gain)
    L, g = oracle.eval_loss_grad(cfg, w.R[i0:i1], w.I[:, i0:i1], th)        # the band as an ordinary sub-image
    local = torch.from_numpy(np.concatenate([L, g[0]]))
    total = sum_over_ranks_in_order(local).numpy()
    full = oracle.RefConfig(w.n, w.n, w.m, sigma0=w.sigma0, gain=w.gain)
    Lf, gf = oracle.eval_loss_grad(full, w.R, w.I, th)
    assert abs(total[0] - Lf[0]) <= 1e-12 * abs(Lf[0]), (total[0], Lf[0])
    assert np.abs(total[1:] - gf[0]).max() <= 1e-10 * np.abs(gf[0]).max()
    dist.destroy_process_group()
    print("band%d-ok" % rank, flush=True)
""")


def test_row_band_sharding_two_ranks_gloo(tmp_path):
    """SURVEY.md 8(e)(2) on CPU: two ranks evaluate row bands of one image pair as ordinary sub-images (the oracle
    stands in for the device call), one small all-gather summed in rank order gives the full loss and gradient."""
    from paper_2104_13715_b200.sharding import row_band
    assert row_band(100, 7, 3, 0) == (0, 32, 0, 38) and row_band(100, 7, 3, 2) == (63, 94, 63, 100)
    with pytest.raises(ValueError):
        row_band(5, 7, 1, 0)
    script = tmp_path / "band_worker.py"
    script.write_text(_BAND_WORKER.format(root=ROOT))
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node=2",
           "--master-addr", "127.0.0.1", "--master-port", str(port), str(script)]
    out = subprocess.run(cmd, capture_output=True, text=True, timeout=240)
    assert out.returncode == 0, out.stdout + out.stderr
    assert "band0-ok" in out.stdout and "band1-ok" in out.stdout, out.stdout


def test_bench_accounting():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.useful_fma(4096, 19, 1) == pytest.approx(1.2007e10, rel=1e-4)
    assert bench.useful_fma(128, 7, 1) == pytest.approx(1.459e6, rel=1e-3)


@pytest.mark.parametrize("m,d", [(5, 0), (7, 0), (11, 3), (13, 0), (15, 2), (19, 0), (19, 3), (27, 0), (33, 1), (41, 0), (47, 3)])
def test_tensor_core_hessian_work_plan(m, d):
    """Host logic of dia_hessian's tensor-core path (dia_hess_tc_plan; no device): the operand slots hold every
    parameter exactly once, every block (gi <= gj) of H is computed by exactly one CTA type, a type's A operand is one
    of the (at most two) groups of its operand tile, and the slots are dealt so that the 32 rows a warp builds read 32
    different shared-memory banks of the staged R tile (kernel pixel (a, b) reads a * pitch + b + const)."""
    import paper_2104_13715_b200 as dia
    G, types, perm = dia.dia_hess_tc_plan(m, d)
    np_ = m * m + (d + 1) * (d + 2) // 2
    assert G == -(-np_ // 128) and perm.shape == (128 * G,)
    assert sorted(perm[perm >= 0].tolist()) == list(range(np_))
    blocks = []
    for g0, g1, a_sel, b_start, nb in types.tolist():
        tile = [g0, g1]
        assert g0 < G and (g1 < G or g1 == 255) and nb in (1, 2) and b_start + nb <= 2 and a_sel in (0, 1)
        gA = tile[a_sel]
        assert gA != 255
        for t in range(b_start, b_start + nb):
            assert tile[t] != 255
            blocks.append((min(gA, tile[t]), max(gA, tile[t])))
    assert sorted(blocks) == [(i, j) for i in range(G) for j in range(i, G)]
    # bank classes: R tile pitch of the fused kernel = RMIN rounded up to 4 (mod 8), RMIN = 48 + round_up(16 + m - 1, 4)
    rmin = 48 + -(-(16 + m - 1) // 4) * 4
    pitch = rmin + ((4 - rmin % 8) + 8) % 8
    conflicts = 0
    for w in range(4 * G):
        rows = [q for q in perm[32 * w:32 * w + 32].tolist() if 0 <= q < m * m]
        banks = [((q // m) * pitch + q % m) % 32 for q in rows]
        conflicts += len(banks) - len(set(banks))
    assert conflicts <= max(2, m * m // 100), conflicts        # the greedy deal leaves at most a few leftovers


def test_tensor_core_hessian_work_plan_errors():
    import paper_2104_13715_b200 as dia
    with pytest.raises(dia.DiaError):
        dia.dia_hess_tc_plan(4, 0)
    with pytest.raises(dia.DiaError):
        dia.dia_hess_tc_plan(7, 9)
