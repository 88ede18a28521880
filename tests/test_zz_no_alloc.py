"""nolsm_gather_submatrix_noalloc against nolsm_gather_submatrix.

Some users of the library cannot let it allocate device memory: a host program whose own pool already owns the whole GPU
(every further cudaMalloc fails), or one that looks at submatrices while long kernels are running (cudaMalloc / cudaFree
wait for the whole device). For them the gather has a second entry point whose scratch is a fixed 16 MiB static device
array inside the library. It must return exactly what the allocating path returns -- a gather does no arithmetic, so the
comparison is bit for bit, the bar of the other gather tests -- and it must do so call after call, although every call
reuses the same array and finds the previous call's matrices in it.

This file is named so that pytest collects it last (`pytest --collect-only`): under `-x` a failure here hides nothing.
Each test builds its own context, so it passes alone in a fresh process (where it is the first use of the static array on
the device) and after the rest of the suite."""
import numpy as np
import pytest
import torch

from workloads import MAT_H, MAT_S, make_system

pytestmark = pytest.mark.gpu


def _ctx(**kw):
    from paper_2205_12182_b200 import Nolsm
    kw.setdefault("timeout_s", 90.0)
    return Nolsm(0, **kw)


def _arrays(s):
    return (torch.from_numpy(s.atom_nb).cuda(), torch.from_numpy(s.row_ptr).cuda(), torch.from_numpy(s.col_idx).cuda(),
            torch.from_numpy(s.fill_np(MAT_H)).cuda(), torch.from_numpy(s.fill_np(MAT_S)).cuda())


def _bits(a):
    a = a.cpu().numpy() if hasattr(a, "cpu") else a
    return np.ascontiguousarray(a).view(np.uint16)


@pytest.mark.parametrize("name,n_atoms,combine", [("cfg0", None, 0), ("cfg2", 300, 0), ("cfg3", 900, 1)])
def test_noalloc_gather_equals_allocating_gather_on_consecutive_calls(name, n_atoms, combine):
    """Back-to-back calls on one stream, largest submatrix first and a smaller one right after it (what the first call left
    in the static array lies beyond and beneath the second call's matrices), both matrices each, into device buffers the
    test owns; then the same atoms again in the opposite order. Every result equals the existing path's bit for bit."""
    s = make_system(name) if n_atoms is None else make_system(name, n_atoms=n_atoms)
    with _ctx(combine=combine) as ctx:
        ctx.assemble(*_arrays(s))
        dims = np.array([ctx.group(i)[2] for i in range(s.n_atoms)])
        order = [int(np.argmax(dims)), int(np.argmin(dims)), int(np.argsort(dims)[len(dims) // 2])]
        assert dims[order[0]] <= 2048 and dims[order[0]] > dims[order[1]]
        want = {(i, w): ctx.gather_submatrix(i, w, fp16=True) for i in order for w in (0, 1)}
        outs = {(i, w): torch.full((int(dims[i]), int(dims[i])), float("nan"), dtype=torch.float16, device="cuda")
                for i in order for w in (0, 1)}
        for i in order + order[::-1]:                       # no synchronisation between the calls: stream order alone
            for w in (0, 1):
                ctx.gather_submatrix_noalloc(i, w, outs[(i, w)])
        torch.cuda.synchronize()
        for key, ref in want.items():
            assert np.array_equal(_bits(outs[key]), _bits(ref)), key
        # host output: the call itself waits for the stream
        i = order[1]
        host = np.full((int(dims[i]), int(dims[i])), np.nan, dtype=np.float16)
        ctx.gather_submatrix_noalloc(i, 1, host)
        assert np.array_equal(_bits(host), _bits(want[(i, 1)]))
    print("noalloc gather", name, "combine", combine, "dims", [int(dims[i]) for i in order])


def test_noalloc_gather_leaves_the_last_result_alone_and_allocates_nothing():
    """Issued while a density-matrix call is in flight (between nolsm_density_matrix and nolsm_energy) it disturbs neither D
    nor E -- it touches neither the workspace nor the outputs -- and the free device memory is the same before and after
    the calls. D and E are compared with the suite's mixed-precision tolerances (atomics make two runs differ in the last
    bits); a clobbered workspace would miss them by orders of magnitude."""
    s = make_system("cfg0")
    nb, rp, ci, Hv, Sv = _arrays(s)
    with _ctx() as ctx:
        ctx.assemble(nb, rp, ci, Hv, Sv)
        D0, D1 = torch.zeros_like(Hv), torch.zeros_like(Hv)
        ctx.density_matrix(s.mu, D0)
        e0 = ctx.energy()
        dim = ctx.group(5)[2]
        out = torch.empty((dim, dim), dtype=torch.float16, device="cuda")
        ctx.gather_submatrix_noalloc(5, 0, out)             # first use on this device in a fresh process: set-up happens here
        torch.cuda.synchronize()
        ctx.density_matrix(s.mu, D1)
        free0 = torch.cuda.mem_get_info()[0]
        for w in (0, 1, 0, 1):
            ctx.gather_submatrix_noalloc(5, w, out)
        torch.cuda.synchronize()
        assert torch.cuda.mem_get_info()[0] == free0
        e1 = ctx.energy()
        assert abs(e1 - e0) <= 1e-3 * abs(e0) and float((D0 - D1).abs().max()) <= 2e-2
        assert np.array_equal(_bits(out), _bits(ctx.gather_submatrix(5, 1, fp16=True)))


def test_noalloc_gather_refuses_what_does_not_fit():
    """A submatrix beyond NOLSM_NOALLOC_MAX_DIM = 2048 is refused with a message that names the limit; nothing is written."""
    from paper_2205_12182_b200 import NolsmError
    s = make_system("pn-14-8.5", n_atoms=1024)
    with _ctx() as ctx:
        ctx.assemble(torch.from_numpy(s.atom_nb).cuda(), torch.from_numpy(s.row_ptr).cuda(), torch.from_numpy(s.col_idx).cuda(),
                     s.fill_torch(MAT_H, "cuda"), s.fill_torch(MAT_S, "cuda"))
        dim = ctx.group(100)[2]
        assert dim > 2048
        out = torch.zeros((4, 4), dtype=torch.float16, device="cuda")
        with pytest.raises(NolsmError) as ei:
            ctx.gather_submatrix_noalloc(100, 0, out)
        assert "NOLSM_NOALLOC_MAX_DIM = 2048" in str(ei.value)
        torch.cuda.synchronize()
        assert not out.any()
        for bad in (-1, s.n_atoms):
            with pytest.raises(NolsmError):
                ctx.gather_submatrix_noalloc(bad, 0, out)
