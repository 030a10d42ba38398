"""CPU-side checks of the boundary: the library loads, exports every symbol include/tddft.h declares, its host logic
(G-vector enumeration, argument checks) agrees with the oracle, and it refuses to run without a GPU."""
import math
import os
import re

import numpy as np
import pytest

from oracle import lattice as olat

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def binding():
    from paper_2309_03513_b200 import build
    build.build(verbose=False)
    from paper_2309_03513_b200 import binding as b
    return b


def test_every_declared_symbol_is_exported(binding):
    hdr = open(os.path.join(ROOT, "include", "tddft.h")).read()
    declared = set(re.findall(r"\b(tddft_[a-z_0-9]+)\s*\(", hdr))
    declared -= {"tddft_options", "tddft_stats"}
    assert declared, "no declarations found"
    for name in sorted(declared):
        assert hasattr(binding._lib, name), "missing export " + name
    assert declared == set(binding.EXPORTS)


def test_options_struct_layout_matches_header(binding):
    # the binding's ctypes mirror must have the fields of the C struct, in order
    hdr = open(os.path.join(ROOT, "include", "tddft.h")).read()
    body = hdr[hdr.index("typedef struct {", hdr.index("All fields optional")):]
    body = body[:body.index("} tddft_options;")]
    body = re.sub(r"/\*.*?\*/", "", body, flags=re.S)
    names = re.findall(r"\b([a-z_0-9]+);", body)
    assert names == [f[0] for f in binding.tddft_options._fields_]


def test_stats_struct_layout_matches_header(binding):
    hdr = open(os.path.join(ROOT, "include", "tddft.h")).read()
    body = hdr[hdr.index("typedef struct {", hdr.index("Counters of the last tddft_apply_liouville call")):]
    body = body[:body.index("} tddft_stats;")]
    body = re.sub(r"/\*.*?\*/", "", body, flags=re.S)
    names = []
    for decl in body.replace("typedef struct {", "").split(";"):
        decl = decl.strip()
        if decl:
            names += [n.strip() for n in re.sub(r"^(long long|double|int)\s+", "", decl).split(",")]
    assert names == [f[0] for f in binding.tddft_stats._fields_]


HEX = [[36.9, 0, 0], [-18.45, 36.9 * math.sqrt(3) / 2, 0], [0, 0, 19.5]]


@pytest.mark.parametrize("lattice,ecut,npwh", [
    (np.eye(3) * 10.0, 10.0, 258), (np.eye(3) * 13.48, 25.0, 2593), (np.eye(3) * 20.2, 25.0, 8683), (HEX, 20.0, 17345),
    ([[4.0, 0, 0], [0.5, 4.2, 0], [0.3, -0.2, 4.5]], 30.0, None),
])
def test_library_and_oracle_build_the_same_g_list(binding, lattice, ecut, npwh):
    m, g2 = binding.tddft_enumerate_gvectors(lattice, ecut)
    mo, go = olat.enumerate_half_sphere(lattice, ecut)
    if npwh is not None:
        assert len(m) == npwh          # SURVEY 8.0 exact enumerations
    assert np.array_equal(m, mo)
    assert np.allclose(g2, go, rtol=1e-13, atol=0)


def test_argument_errors_and_no_gpu_behaviour(binding):
    import ctypes as C
    lib = binding._lib
    n = C.c_long(0)
    assert lib.tddft_enumerate_gvectors(None, C.c_double(1.0), C.c_long(0), None, None, C.byref(n)) == binding.TDDFT_EINVAL
    lat = np.eye(3).reshape(9) * 10.0
    miller = np.zeros(3, dtype=np.int32)
    rc = lib.tddft_enumerate_gvectors(lat.ctypes.data_as(C.c_void_p), C.c_double(10.0), C.c_long(1),
                                      miller.ctypes.data_as(C.c_void_p), None, C.byref(n))
    assert rc == binding.TDDFT_EINVAL and n.value == 258        # capacity too small, count still reported
    h = C.c_void_p(None)
    assert lib.tddft_init(C.byref(h), None, None, C.c_double(1.0), 1, None, None, None, None, None, C.c_double(0.1), None) == binding.TDDFT_EINVAL
    assert h.value is None
    assert lib.tddft_apply_liouville(None, None, None, 1, 0) == binding.TDDFT_EINVAL
    assert lib.tddft_destroy(None) == binding.TDDFT_OK
    try:
        import torch
        has_gpu = torch.cuda.is_available()
    except Exception:
        has_gpu = False
    if not has_gpu:
        # the product path fails loudly without a device: no CPU fallback
        grid = (C.c_int * 3)(24, 24, 24)
        nocc = (C.c_int * 2)(1, 0)
        dummy = np.zeros(600)
        rc = lib.tddft_init(C.byref(h), lat.ctypes.data_as(C.c_void_p), grid, C.c_double(10.0), 1, nocc,
                            dummy.ctypes.data_as(C.c_void_p), None, dummy.ctypes.data_as(C.c_void_p), None, C.c_double(0.25), None)
        assert rc == binding.TDDFT_ECUDA
        assert "no CUDA device" in binding.tddft_last_error()


def test_bench_sharding_two_ranks_gloo(tmp_path):
    """The N > 1 path shards independent trial-vector blocks over ranks (no data-path collective): with gloo on CPU,
    two ranks must draw different blocks from the same orbitals and agree on the max-over-ranks time reduction."""
    import subprocess
    import sys
    script = tmp_path / "two_ranks.py"
    script.write_text('''
import os, sys
sys.path.insert(0, %r)
import numpy as np, torch, torch.distributed as dist
import synthetic_inputs as inputs
from oracle import lattice as olat
dist.init_process_group("gloo")
rank, world = dist.get_rank(), dist.get_world_size()
cfg = inputs.config(1)
miller, g2 = olat.enumerate_half_sphere(cfg["lattice"], cfg["ecut"])
inp = inputs.make_problem_inputs(cfg, g2)
inp["rng"] = np.random.Generator(np.random.PCG64(cfg["seed"] + 1000 * (rank + 1)))
X = inputs.make_trial_block(cfg, inp, 2, 0)
psi_sum = torch.tensor([float(np.abs(inp["psi"][0]).sum())], dtype=torch.float64)
x_sum = torch.tensor([float(np.abs(X).sum())], dtype=torch.float64)
allpsi = [torch.zeros_like(psi_sum) for _ in range(world)]; allx = [torch.zeros_like(x_sum) for _ in range(world)]
dist.all_gather(allpsi, psi_sum); dist.all_gather(allx, x_sum)
assert allpsi[0].item() == allpsi[1].item(), "orbitals must be identical on every rank"
assert allx[0].item() != allx[1].item(), "each rank must own a different trial-vector block"
t = torch.tensor([10.0 + rank], dtype=torch.float64)
dist.all_reduce(t, op=dist.ReduceOp.MAX)
assert t.item() == 11.0
dist.destroy_process_group()
print("ok", rank)
''' % ROOT)
    r = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node=2",
                        "--master-addr", "127.0.0.1", "--master-port", "29617", str(script)],
                       capture_output=True, text=True, timeout=300)
    assert r.returncode == 0, r.stdout + r.stderr


def test_sharded_apply_collective_two_ranks_gloo(tmp_path):
    """The one exchange step of the sharded apply (binding.allreduce_sum_, used by tddft_apply_liouville_sharded): with gloo on CPU
    tensors and world size 2 the partial results are summed on every rank, complex tensors through their real view."""
    import subprocess, sys, textwrap
    script = tmp_path / "w.py"
    script.write_text(textwrap.dedent("""
        import os, sys, torch, torch.distributed as dist
        sys.path.insert(0, %r)
        from paper_2309_03513_b200 import binding as b
        dist.init_process_group("gloo")
        r = dist.get_rank()
        t = torch.full((3, 5), complex(r + 1.0, -(r + 1.0)), dtype=torch.complex128)
        b.allreduce_sum_(t)
        assert torch.allclose(t, torch.full((3, 5), complex(3.0, -3.0), dtype=torch.complex128)), t
        dist.destroy_process_group()
    """ % str(ROOT)))
    env = dict(os.environ, MASTER_ADDR="127.0.0.1", MASTER_PORT="29613")
    r = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr", "127.0.0.1",
                        "--master-port", "29613", str(script)], capture_output=True, text=True, env=env, timeout=300)
    assert r.returncode == 0, r.stdout + r.stderr
