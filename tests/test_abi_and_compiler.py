"""CPU-only checks of the boundary and the host DAG compiler: the shared library loads and exports every symbol
include/cos.h declares, argument errors come back as status codes, and the compiled DAG (COS_BUILD_HOST_ONLY: no
CUDA call) has the structure the paper fixes (3^n masks, 2^n - 1 readouts, readout layers, Lemma 2) and the R-form
sizes of SURVEY.md 8(a).  No compute call is made here."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def cos():
    from paper_2507_12349_b200 import build as b
    b.build()
    import paper_2507_12349_b200 as cos_mod
    cos_mod.load_library()
    return cos_mod


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "cos.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(cos_[a-z0-9_]+)\s*\(", text)))


def test_library_exports_every_declared_symbol(cos):
    lib = ctypes.CDLL(cos.lib_path())
    names = declared_symbols()
    assert "cos_build" in names and "cos_eval" in names and "cos_free" in names and len(names) >= 14
    for name in names:
        assert hasattr(lib, name), name
    assert sorted(cos.EXPORTS) == names          # the binding wraps exactly the declared entry points


def test_argument_errors_are_status_codes(cos):
    for args in [(0, 2, 0, None, 0), (13, 2, 0, None, 0), (4, 0, 0, None, 0), (4, 2, 7, None, 0), (4, 2, 0, None, 3),
                 (4, 5, 0, [0.1] * 5, 0)]:
        with pytest.raises(cos.CosError) as ei:
            cos.cos_build_ex(*args, flags=cos.COS_BUILD_HOST_ONLY)
        assert ei.value.code in (cos.COS_EINVAL, cos.COS_EUNSUPPORTED)
        assert cos.cos_last_error()
    cos.cos_free(None)                           # no-op by contract


def test_no_cpu_fallback(cos):
    """Without a CUDA device cos_build must fail loudly; a host-only handle refuses to evaluate."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("CPU-box check")
    with pytest.raises(cos.CosError) as ei:
        cos.cos_build(4, 2, 0, None, 0)
    assert ei.value.code == cos.COS_ECUDA
    h = cos.cos_build_ex(4, 2, 0, None, 0, flags=cos.COS_BUILD_HOST_ONLY)
    lib = cos.load_library()
    rc = lib.cos_eval(h, ctypes.c_void_p(8), 1, ctypes.c_void_p(8), None)
    assert rc == cos.COS_ECUDA
    cos.cos_free(h)


SIZES = [  # (n, nf, lattice, shifts, all_subsets) -> (states, edges, readout edges, max layer): SURVEY.md 8(a) [probe]
    ((4, 2, 0, None, False), (191, 522, 13, 49)),
    ((8, 2, 0, None, True), (61353, 313828, 3839, 10517)),
    ((10, 2, 0, None, False), (589979, 3913410, 91, 95353)),
    ((10, 2, 0, None, True), (815831, 5212505, 24063, 126237)),
    ((10, 3, 0, (0.2, 0.0, -0.2), False), (1769937, 16020777, 273, 286059)),
    ((6, 3, 0, (0.2, 0.0, -0.2), False), (9465, 59205, None, 1983)),
    ((6, 2, 1, (0.3, -0.3), False), (67524, 465976, None, 15344)),
    ((5, 2, 0, None, False), (795, 2699, None, 177)),
]


@pytest.mark.parametrize("args,want", SIZES)
def test_rform_sizes(cos, args, want):
    n, nf, lat, sh, allsub = args
    h = cos.cos_build_ex(n, nf, lat, sh, n if allsub else 0, flags=cos.COS_BUILD_HOST_ONLY)
    try:
        info = cos.dag_summary(h)
        got = (info["n_states"], info["n_edges"], info["n_readout_edges"], info["max_layer_states"])
        for g, w in zip(got, want):
            assert w is None or g == w, (got, want)
        assert info["n_layers"] == 2 * n
        assert sum(info["layer_states"]) == info["n_states"]
    finally:
        cos.cos_free(h)


def test_structure_fixed_by_the_paper(cos):
    """3^n masks minus the unreachable ones never exceeds 3^n; all-subset readouts are 2^n - 1
    (PAPER.md:156); n = 4 per-layer state counts of SURVEY.md 8(a); single-output uses only root 0."""
    n = 4
    h1 = cos.cos_build_ex(n, 2, 0, None, 0, flags=cos.COS_BUILD_HOST_ONLY)
    h2 = cos.cos_build_ex(n, 2, 0, None, n, flags=cos.COS_BUILD_HOST_ONLY)
    try:
        i1, i2 = cos.dag_summary(h1), cos.dag_summary(h2)
        assert i1["layer_states"] == [1, 4, 15, 33, 46, 49, 30, 13]
        assert i2["layer_states"] == [4, 10, 26, 49, 57, 56, 30, 13]
        assert i1["n_out"] == 1 and i2["n_out"] == 2 ** n - 1
        assert i2["n_masks"] <= 3 ** n and i1["n_masks"] <= 3 ** n
        assert i2["n_readout_edges"] == 4 + 18 + 28 + 13
        assert i1["n_states_unpruned"] >= i1["n_states"]
    finally:
        cos.cos_free(h1)
        cos.cos_free(h2)


def test_sb_colour_scaling(cos):
    """SB mode carries the colour in the state: states = N_f x (uniform states) for the same lattice / readout, and
    shift edges exist only with shifts (Eq. 79-80)."""
    hu = cos.cos_build_ex(6, 3, 0, None, 0, flags=cos.COS_BUILD_HOST_ONLY)
    hs = cos.cos_build_ex(6, 3, 0, (0.1, 0.2, 0.3), 0, flags=cos.COS_BUILD_HOST_ONLY)
    try:
        iu, is_ = cos.dag_summary(hu), cos.dag_summary(hs)
        assert is_["n_states"] == 3 * iu["n_states"]
        assert is_["n_blocks"] == 3 and iu["n_blocks"] == 1
        assert is_["n_edges"] > 3 * iu["n_edges"]        # + E3 and the colour fan-out of E4
    finally:
        cos.cos_free(hu)
        cos.cos_free(hs)


def test_det_route_argument_checks_need_no_gpu(cos):
    """cos_det_workspace_bytes is pure arithmetic; cos_det_eval validates its arguments before touching CUDA."""
    lib = cos.load_library()
    n, nb, B = 10, 3, 8192
    assert cos.cos_det_workspace_bytes(n, nb, cos.COS_DET_FP64, B) == 8 * (nb + 2) * 2 ** n * B + 4 * 2 ** n
    assert cos.cos_det_workspace_bytes(n, nb, cos.COS_DET_DD, B) == 16 * (nb + 2) * 2 ** n * B + 4 * 2 ** n
    assert cos.cos_det_workspace_bytes(n, 4, 0, B) == -1 and cos.cos_det_workspace_bytes(n, nb, 0, -1) == -1
    p = ctypes.c_void_p(256)
    for args, code in (((0, 3, 3, 0, None, 0, p, 4, p, p, 1 << 30, None), cos.COS_EINVAL),            # n
                       ((4, 5, 5, 0, None, 0, p, 4, p, p, 1 << 30, None), cos.COS_EUNSUPPORTED),      # flavours
                       ((4, 3, 2, 0, None, 0, p, 4, p, p, 1 << 30, None), cos.COS_EINVAL),            # blocks
                       ((4, 3, 3, 2, None, 0, p, 4, p, p, 1 << 30, None), cos.COS_EINVAL),            # lattice
                       ((4, 3, 3, 0, None, 5, p, 4, p, p, 1 << 30, None), cos.COS_EINVAL),            # precision
                       ((4, 3, 3, 0, None, 0, None, 4, p, p, 1 << 30, None), cos.COS_EINVAL),         # NULL input
                       ((4, 3, 3, 0, None, 1, p, 4, p, ctypes.c_void_p(264), 1 << 30, None), cos.COS_EINVAL),   # alignment
                       ((4, 3, 3, 0, None, 0, p, 4, p, p, 64, None), cos.COS_EINVAL)):                # workspace size
        assert lib.cos_det_eval(*args) == code, args
        assert cos.cos_last_error()
    assert lib.cos_det_eval(4, 3, 3, 0, None, 0, p, 0, p, p, 0, None) == cos.COS_OK                  # batch 0: no-op


def test_structural_limits_are_unsupported_not_out_of_memory(cos):
    """include/cos.h, cos_build: structural limits come back as COS_EUNSUPPORTED with the reason, COS_ENOMEM is memory
    exhaustion only.  Honeycomb SB-CoS at n = 11 exceeds the 24-bit destination index of the layer program (north_star
    asks for orders up to 12 on both lattices: the honeycomb range of this build ends at n = 10 for SB-CoS; the uniform
    honeycomb DAG still compiles at n = 11)."""
    with pytest.raises(cos.CosError) as ei:
        cos.cos_build_ex(11, 2, cos.COS_LATTICE_HONEYCOMB, [0.3, -0.3], 0, flags=cos.COS_BUILD_HOST_ONLY)
    assert ei.value.code == cos.COS_EUNSUPPORTED and "24-bit" in str(ei.value)
    with pytest.raises(cos.CosError) as ei:
        cos.cos_build_ex(4, 5, cos.COS_LATTICE_SQUARE, [0.1] * 5, 0, flags=cos.COS_BUILD_HOST_ONLY)
    assert ei.value.code == cos.COS_EUNSUPPORTED
    # the largest BASELINE-shaped honeycomb order this build supports compiles host-only (3.9e7 states)
    h = cos.cos_build_ex(10, 2, cos.COS_LATTICE_HONEYCOMB, [0.3, -0.3], 0, flags=cos.COS_BUILD_HOST_ONLY)
    assert cos.cos_info(h, "n_states") == 39320580 and cos.cos_info(h, "device") == -1
    cos.cos_free(h)


def test_tuning_and_reserve_argument_checks(cos):
    """cos_set_tuning / cos_reserve on a host-only handle: value checks are status codes; nothing touches CUDA."""
    h = cos.cos_build_ex(5, 2, cos.COS_LATTICE_SQUARE, None, 0, flags=cos.COS_BUILD_HOST_ONLY)
    try:
        for what, good, bad in (("prefetch", 16, -1), ("prefetch", 0, 5000), ("warps_per_cta", 8, 0),
                                ("warps_per_cta", 24, 25), ("blocks_per_cta_cap", 0, 70000), ("host_slices", 8, 9),
                                ("host_slices", 1, 0), ("tiles_per_chunk", 0, -2)):
            cos.cos_set_tuning(h, what, good)
            with pytest.raises(cos.CosError) as ei:
                cos.cos_set_tuning(h, what, bad)
            assert ei.value.code == cos.COS_EINVAL
        cos.cos_set_tuning(h, "pdl", 0)
        cos.cos_set_tuning(h, "fused", 1)
        assert cos.cos_info(h, "fused") == 0            # host-only handles have no fused path
        with pytest.raises(cos.CosError) as ei:
            cos.cos_set_tuning(h, 42, 1)
        assert ei.value.code == cos.COS_EINVAL
        with pytest.raises(cos.CosError) as ei:
            cos.cos_reserve(h, 64)
        assert ei.value.code == cos.COS_ECUDA
        with pytest.raises(cos.CosError) as ei:
            cos.cos_reserve(h, -1)
        assert ei.value.code == cos.COS_EINVAL
    finally:
        cos.cos_free(h)


def test_library_reads_no_environment_variable(cos):
    """The launch tuning goes through cos_set_tuning only (include/cos.h): no getenv in the product sources."""
    csrc = os.path.join(ROOT, "paper_2507_12349_b200", "csrc")
    for name in os.listdir(csrc):
        assert "getenv" not in open(os.path.join(csrc, name)).read(), name


def test_host_compiler_under_address_and_ub_sanitizers(tmp_path):
    """g++ -fsanitize=address,undefined on the host DAG compiler, every mode, n = 1..8 (tests/host_compiler_sanitize.cpp):
    no report, exit code 0."""
    import subprocess
    exe = str(tmp_path / "host_compiler_sanitize")
    subprocess.check_call(["g++", "-O1", "-g", "-std=c++17", "-fsanitize=address,undefined", "-fno-sanitize-recover=undefined",
                           "-o", exe, os.path.join(ROOT, "tests", "host_compiler_sanitize.cpp"),
                           os.path.join(ROOT, "paper_2507_12349_b200", "csrc", "cos_compile.cpp")])
    r = subprocess.run([exe], capture_output=True, text=True, timeout=600)
    assert r.returncode == 0 and r.stdout.startswith("ok,") and not r.stderr.strip(), r.stdout + r.stderr


def test_future_and_past_equivalence_classes(cos):
    """Compiler compression, PAPER.md:219-241 (Eq. 25-28), evaluated on the reduced recurrence (cos_equivalence_stats):
    with propagator entries compared as symbols NO two states of a layer share a future signature (the closing factor
    G_lambda[e][h] and the continuation factors G_lambda[e][j] pin colour, endpoint, head and mask), and the only past
    equivalences are the N_c fresh-head states of a close-and-open step (Eq. 12, 70-71: equal in-edges for every colour)
    and the initial states (value 1, Eq. 66) -- both already exploited by the kernel (one closing sum fanned out to the
    N_c states; edge count after the past merge = the executed multiply-adds before E2/E4 coalescing)."""
    sb3 = [0.2, 0.0, -0.2]
    for args in [(4, 2, 0, None, 0), (6, 2, 0, None, 0), (8, 2, 0, None, 0), (5, 3, 0, None, 0)]:
        r = cos.cos_equivalence_stats(*args)
        h = cos.cos_build_ex(*args, flags=cos.COS_BUILD_HOST_ONLY)
        assert r["states"] == cos.cos_info(h, "n_states")
        assert r["edges"] == cos.cos_info(h, "n_edges") + cos.cos_info(h, "n_readout_edges")
        cos.cos_free(h)
        assert r["future_classes"] == r["states"] and r["edges_after_future_merge"] == r["edges"]
        assert r["past_classes"] == r["states"] and r["edges_after_past_merge"] == r["edges"]      # uniform, one root
    r = cos.cos_equivalence_stats(4, 2, 0, None, 4)            # all subsets: the 4 initial states (roots 0..3) are equal
    assert r["future_classes"] == r["states"] == 245 and r["past_classes"] == 242
    for n, want_states, want_past in ((6, 9465, 9041), (8, 135213, 131093)):
        r = cos.cos_equivalence_stats(n, 3, 0, sb3, 0)
        assert r["states"] == want_states and r["future_classes"] == want_states
        assert r["past_classes"] == want_past and r["edges_after_past_merge"] < r["edges"]
    r = cos.cos_equivalence_stats(4, 2, 1, [0.3, -0.3], 0)     # honeycomb, sublattice labels in the mask
    assert r["future_classes"] == r["states"] == 2292 and r["past_classes"] == 2233
    r = cos.cos_equivalence_stats(5, 3, 0, [0.4], 0, flags=cos.COS_BUILD_UNIFORM_SHIFT)
    assert r["future_classes"] == r["states"] == r["past_classes"]
    # the fresh-head coefficient -N_f is kept as a full integer in the signature: many flavours (uniform mode has no upper
    # bound on N_f) must give the same class structure as two flavours, not spurious merges
    base = cos.cos_equivalence_stats(5, 2, 0, None, 0)
    for nf in (9, 40, 100000):
        r = cos.cos_equivalence_stats(5, nf, 0, None, 0)
        assert r == base and r["future_classes"] == r["states"] == r["past_classes"]
    with pytest.raises(cos.CosError):
        cos.cos_equivalence_stats(4, 2, 0, None, 3)
