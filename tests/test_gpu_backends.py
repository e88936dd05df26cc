"""GPU parity of the alternative back ends of sm_sign_ns that the library selects by size or that the
environment forces (each in its own process: the selection is read once per process):
  SM_UMMA_NCTA=1|2   one CTA / two CTAs per tile of the tcgen05 kernel
  SM_UMMA_MC=1|0     two CTAs: own cta_group::1 MMAs with the B rows multicast / cta_group::2 MMAs with a relayed stage signal
  SM_UMMA_TMAP=1     cta_group::2 MMAs whose operands come through tensor-map TMA signalling the leader's barrier directly
  SM_UMMA_REV=1|0    PHASE 2 walks the tile table backwards / forwards
  SM_UMMA_STAGES=3|4 depth of the operand ring of the single-CTA kernel
  SM_UMMA_DYN=1|0    tiles handed out by a global counter / dealt round robin
  SM_UMMA_STREAM=1   one launch walks every product of every step (dependency counters per group of submatrices)
  SM_UMMA_SLOTS=2|1  submatrices a CTA pair of the fused kernel interleaves
  SM_UMMA_SYM=1|0    symmetric half tiles with mirrored stores / true products with an MN-major B operand
  SM_UMMA_FUSED=1|0  one launch runs every step of a submatrix (k_umma_fused) / one launch per product
  SM_UMMA_RESIDENT=1|0  submatrices with Pd <= 256 iterate inside one SM (k_umma_resident) / grouped tiles for all
  SM_UMMA_LT=0|1     grouped tiles: iterates stored lower-triangular, the upper part read through MN-major descriptors
  SM_UMMA_FOLD=1|0   single-CTA symmetric tiles: a short last row panel is computed as extra columns of the other panels / as a panel
  SM_UMMA_SHAREA=1|0 product 1: a tile that holds its panel's diagonal square reads its A rows from the B stage / loads them
  SM_F64_SIMT=0|1    DMMA tensor tiles (default) / DFMA register tiles
The two-CTA and fused variants exist only in a -DSM_MEASURE build of the library (build.py --measure); their cases
are skipped on the default build.
Each case runs NS steps on a seeded workload whose submatrices span several tiles and ragged tails and
compares with the oracle's NS-k polynomial (exact-arithmetic result of k steps, reading A13)."""
import os
import subprocess
import sys
import textwrap

import pytest

pytestmark = pytest.mark.gpu
pytest.importorskip("torch")

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

SNIPPET = textwrap.dedent("""
    import os, sys, numpy as np, torch
    sys.path.insert(0, {root!r})
    import paper_2205_14741_b200.binding as sm
    from oracle import oracle as orc
    from workloads.generator import make_workload
    x_dtype, pad, k, tol_abs, sym_exact = {x_dtype!r}, {pad}, {k}, {tol_abs}, {sym_exact}
    cache = {cache!r}      # this pytest session's directory of oracle references (several cases share a workload)
    def ns_reference(i, T):
        f = os.path.join(cache, "ns_{n_mol}_{b}_{n_occ}_{cutoff}_%d_%d.npy" % (k, i))
        if os.path.exists(f):
            return np.load(f)
        ref = orc.ns_polynomial(T, orc.gershgorin(T), k)
        np.save(f + ".tmp.npy", ref); os.replace(f + ".tmp.npy", f)
        return ref
    wl = make_workload({n_mol}, {b}, {n_occ}, {cutoff}, seed=33)
    A = sm.Bcsr(wl); P = sm.sm_build_pattern(A, pad); Ph = sm.pattern_to_host(P)
    cols, col_off, n = sm.sm_plan_columns(P, None)
    X, scale = sm.sm_gather(A, P, cols, col_off, n, 0.0, "gershgorin", x_dtype)
    iters, res = sm.sm_sign_ns(P, cols, col_off, n, P.packed_elems, x_dtype, X, k, 0.0)
    torch.cuda.synchronize()
    assert (iters == k).all()
    dims = Ph.dim
    picks = set([int(np.argmin(dims)), int(np.argmax(dims)), 0, wl.n_blk // 2])
    for pdv in np.unique(Ph.dim_pad):                      # one column of every padded size (every tile shape)
        idx = np.nonzero(Ph.dim_pad == pdv)[0]
        picks.add(int(idx[0])); picks.add(int(idx[np.argmax(dims[idx])]))
    picks = sorted(picks)
    def img_index(Pd):
        r = np.arange(Pd)[:, None]; c = np.arange(Pd)[None, :]
        return (c >> 6) * Pd * 64 + r * 64 + ((((c & 63) >> 3) ^ (r & 7)) << 3) + (c & 7)
    worst = 0.0
    for i in picks:
        T = orc.gather(wl, i); m = T.shape[0]; Pd = int(Ph.dim_pad[i]); lo = int(Ph.sub_off[i])
        buf = X[lo:lo + Pd * Pd].double().cpu().numpy()
        x = buf[img_index(Pd)] if x_dtype in ("bf16", "f16") else buf.reshape(Pd, Pd)
        ref = ns_reference(i, T)
        err = np.abs(x[:m, :m] - ref).max(); worst = max(worst, err)
        assert err <= tol_abs, (i, m, err)
        assert not x[m:].any() and not x[:, m:].any(), "padding must stay zero"
        if sym_exact:
            assert np.array_equal(x, x.T), "iterate must be exactly symmetric"
        else:
            assert np.abs(x - x.T).max() <= tol_abs
    print("OK dims", int(dims.min()), int(dims.max()), "pads", sorted(set(int(x) for x in Ph.dim_pad)), "worst", worst)
""")

M = "measure"      # case needs a -DSM_MEASURE build
CASES = [
    # env, x_dtype, pad, (n_mol, b, n_occ, cutoff), steps, tolerance (max-abs vs the NS-k polynomial), exact symmetry, build
    ({"SM_UMMA_NCTA": "1", "SM_UMMA_SYM": "1"}, "bf16", 64, (90, 23, 4, 5.0), 3, 2.5e-2, True, None),
    ({"SM_UMMA_DYN": "0"}, "f16", 64, (90, 23, 4, 5.0), 3, 3e-3, True, None),
    ({"SM_UMMA_FOLD": "0"}, "f16", 64, (90, 23, 4, 5.0), 3, 3e-3, True, None),
    ({"SM_UMMA_SHAREA": "0"}, "f16", 64, (90, 23, 4, 5.0), 3, 3e-3, True, None),
    ({"SM_UMMA_SHAREA": "0", "SM_UMMA_RESIDENT": "0"}, "bf16", 64, (300, 6, 3, 6.0), 3, 2.5e-2, True, None),
    ({"SM_UMMA_FOLD": "0", "SM_UMMA_RESIDENT": "0"}, "bf16", 64, (300, 6, 3, 6.0), 3, 2.5e-2, True, None),
    ({"SM_UMMA_FOLD": "1", "SM_UMMA_RESIDENT": "0"}, "f16", 64, (300, 6, 3, 6.0), 5, 3e-3, True, None),
    ({"SM_UMMA_FOLD": "1", "SM_UMMA_STREAM": "1", "SM_UMMA_RESIDENT": "0"}, "f16", 64, (300, 6, 3, 6.0), 4, 3e-3, True, None),
    ({"SM_UMMA_STREAM": "1"}, "f16", 64, (90, 23, 4, 5.0), 4, 3e-3, True, None),
    ({"SM_UMMA_SYM": "0"}, "f16", 64, (90, 23, 4, 5.0), 3, 3e-3, False, None),
    ({"SM_UMMA_SYM": "0"}, "bf16", 64, (300, 6, 3, 6.0), 3, 2.5e-2, False, None),
    # shared-memory-resident kernel: every padded size 64 .. 256 plus larger ones through the grouped path in one call
    ({"SM_UMMA_RESIDENT": "1"}, "bf16", 64, (300, 6, 3, 6.0), 3, 2.5e-2, True, None),
    ({"SM_UMMA_RESIDENT": "1"}, "f16", 64, (300, 6, 3, 6.0), 5, 3e-3, True, None),
    ({"SM_UMMA_RESIDENT": "1"}, "f16", 64, (40, 6, 3, 4.0), 4, 3e-3, True, None),
    ({"SM_UMMA_RESIDENT": "1"}, "bf16", 64, (60, 23, 4, 3.2), 3, 2.5e-2, True, None),
    ({"SM_UMMA_RESIDENT": "0"}, "f16", 64, (300, 6, 3, 6.0), 5, 3e-3, True, None),
    # staged epilogue (bulk stores) and "128-lower" storage with transposed (MN-major) operand reads
    ({"SM_UMMA_EPI": "1"}, "bf16", 64, (90, 23, 4, 5.0), 3, 2.5e-2, True, None),
    ({"SM_UMMA_EPI": "1", "SM_UMMA_RESIDENT": "0"}, "f16", 64, (300, 6, 3, 6.0), 5, 3e-3, True, None),
    ({"SM_UMMA_EPI": "1", "SM_UMMA_LT": "1"}, "bf16", 64, (90, 23, 4, 5.0), 3, 2.5e-2, True, None),
    ({"SM_UMMA_EPI": "1", "SM_UMMA_LT": "1", "SM_UMMA_RESIDENT": "0"}, "f16", 64, (300, 6, 3, 6.0), 5, 3e-3, True, None),
    ({"SM_UMMA_EPI": "1", "SM_UMMA_LT": "1"}, "f16", 64, (40, 23, 4, 8.0), 4, 3e-3, True, None),
    ({"SM_UMMA_FUSED": "0", "SM_UMMA_NCTA": "2", "SM_UMMA_SYM": "1", "SM_UMMA_MC": "1"}, "bf16", 64, (90, 23, 4, 5.0), 3, 2.5e-2, True, M),
    ({"SM_UMMA_FUSED": "0", "SM_UMMA_NCTA": "2", "SM_UMMA_SYM": "1", "SM_UMMA_MC": "0"}, "bf16", 64, (90, 23, 4, 5.0), 3, 2.5e-2, True, M),
    ({"SM_UMMA_FUSED": "0", "SM_UMMA_NCTA": "2", "SM_UMMA_SYM": "1", "SM_UMMA_MC": "1", "SM_UMMA_REV": "0"}, "f16", 64, (90, 23, 4, 5.0), 3, 3e-3, True, M),
    ({"SM_UMMA_FUSED": "0", "SM_UMMA_NCTA": "2", "SM_UMMA_SYM": "1", "SM_UMMA_MC": "0"}, "f16", 64, (90, 23, 4, 5.0), 4, 3e-3, True, M),
    ({"SM_UMMA_FUSED": "0", "SM_UMMA_NCTA": "2", "SM_UMMA_SYM": "0"}, "bf16", 64, (90, 23, 4, 5.0), 3, 2.5e-2, False, M),
    ({"SM_UMMA_FUSED": "1"}, "bf16", 64, (90, 23, 4, 5.0), 3, 2.5e-2, True, M),
    ({"SM_UMMA_FUSED": "1", "SM_UMMA_SLOTS": "1"}, "bf16", 64, (90, 23, 4, 5.0), 4, 2.5e-2, True, M),
    ({"SM_UMMA_FUSED": "1"}, "f16", 64, (90, 23, 4, 5.0), 4, 3e-3, True, M),
    ({"SM_F64_SIMT": "0"}, "f64", 4, (90, 23, 4, 5.0), 4, 1e-13, True, None),
    ({"SM_F64_SIMT": "1"}, "f64", 16, (90, 23, 4, 5.0), 4, 1e-13, False, None),
]


def _measure_build():
    import paper_2205_14741_b200.binding as sm
    return bool(sm.build_info() & 1)


@pytest.fixture(scope="module")
def ref_cache(tmp_path_factory):
    return str(tmp_path_factory.mktemp("ns_refs"))


@pytest.mark.parametrize("env,x_dtype,pad,wl,k,tol_abs,sym_exact,need", CASES)
def test_backend_matches_ns_polynomial(env, x_dtype, pad, wl, k, tol_abs, sym_exact, need, ref_cache):
    if need == M and not _measure_build():
        pytest.skip("variant exists only in a -DSM_MEASURE build (build.py --measure)")
    n_mol, b, n_occ, cutoff = wl
    code = SNIPPET.format(root=ROOT, x_dtype=x_dtype, pad=pad, k=k, tol_abs=tol_abs, sym_exact=sym_exact,
                          n_mol=n_mol, cutoff=cutoff, b=b, n_occ=n_occ, cache=ref_cache)
    e = dict(os.environ)
    e.update(env)
    p = subprocess.run([sys.executable, "-c", code], env=e, capture_output=True, text=True, timeout=600, cwd=ROOT)
    assert p.returncode == 0, p.stdout[-2000:] + p.stderr[-4000:]
    assert "OK dims" in p.stdout


HASH_SNIPPET = textwrap.dedent("""
    import sys, hashlib, numpy as np, torch
    sys.path.insert(0, {root!r})
    import paper_2205_14741_b200.binding as sm
    from workloads.generator import make_workload
    wl = make_workload(200, 23, 4, 5.0, seed=34)
    A = sm.Bcsr(wl); P = sm.sm_build_pattern(A, 64)
    cols, col_off, n = sm.sm_plan_columns(P, P.order)
    X, scale = sm.sm_gather(A, P, cols, col_off, n, 0.0, "global", "bf16")
    iters, res = sm.sm_sign_ns(P, cols, col_off, n, P.packed_elems, "bf16", X, 7, 0.0)
    torch.cuda.synchronize()
    assert (iters == 7).all() and bool(torch.isfinite(X.float()).all())
    r = res.cpu().numpy()
    print("HASH", hashlib.sha1(X.view(torch.int16).cpu().numpy().tobytes()).hexdigest(), repr(float(r.sum())), repr(float(r.max())))
""")

SYM_VARIANTS = [
    {"SM_UMMA_RESIDENT": "0"},
    {"SM_UMMA_RESIDENT": "0", "SM_UMMA_SHAREA": "0"},
    {"SM_UMMA_RESIDENT": "0", "SM_UMMA_REV": "0"},
    {"SM_UMMA_RESIDENT": "0", "SM_UMMA_STAGES": "3"},
    {"SM_UMMA_RESIDENT": "0", "SM_UMMA_DYN": "0"},
    {"SM_UMMA_RESIDENT": "0", "SM_UMMA_DYN": "0", "SM_UMMA_STAGES": "3"},
    {"SM_UMMA_RESIDENT": "0", "SM_UMMA_STREAM": "1"},
    {"SM_UMMA_RESIDENT": "0", "SM_UMMA_EPI": "1"},
    {"SM_UMMA_RESIDENT": "0", "SM_UMMA_EPI": "1", "SM_UMMA_DYN": "0"},
    {"SM_UMMA_RESIDENT": "0", "SM_UMMA_EPI": "1", "SM_UMMA_LT": "1"},
    {"SM_UMMA_RESIDENT": "0", "SM_UMMA_EPI": "1", "SM_UMMA_STREAM": "1"},
]
# (SM_UMMA_RESIDENT=0 like the list above: the resident kernel adds X after the accumulation instead of through identity
# MMAs inside it, so the few submatrices with Pd <= 256 of this workload would differ from the grouped tiles in the last bit)
SYM_VARIANTS_MEASURE = [
    {"SM_UMMA_RESIDENT": "0", "SM_UMMA_FUSED": "0", "SM_UMMA_NCTA": "2", "SM_UMMA_MC": "1"},
    {"SM_UMMA_RESIDENT": "0", "SM_UMMA_FUSED": "0", "SM_UMMA_NCTA": "2", "SM_UMMA_MC": "0"},
    {"SM_UMMA_RESIDENT": "0", "SM_UMMA_FUSED": "0", "SM_UMMA_NCTA": "2", "SM_UMMA_MC": "0", "SM_UMMA_TMAP": "1"},
    {"SM_UMMA_RESIDENT": "0", "SM_UMMA_FUSED": "0", "SM_UMMA_NCTA": "2", "SM_UMMA_MC": "0", "SM_UMMA_TMAP": "1", "SM_UMMA_STAGES": "3"},
    {"SM_UMMA_FUSED": "1", "SM_UMMA_SLOTS": "1"},
    {"SM_UMMA_FUSED": "1", "SM_UMMA_SLOTS": "2"},
]


def test_symmetric_tile_variants_are_bit_identical():
    """Every SYM variant (one CTA, two CTAs with multicast or relay, either walk direction, fused with one or two
    slots) issues the same MMAs per output element in the same k order and applies the same epilogue arithmetic, so
    7 odd-count steps (copy-back path) on 200 submatrices spanning several tile shapes give the same bits; the
    fused residual is the same to rounding of its fixed-order partial sums (grouped per tile and warp)."""
    seen = {}
    for env in SYM_VARIANTS + (SYM_VARIANTS_MEASURE if _measure_build() else []):
        e = dict(os.environ)
        # the folded geometry (default) takes the last rows of a submatrix from the TRANSPOSED tile elements: equal in
        # exact arithmetic, not to the bit (X Wh is symmetric only because X and Wh commute); it has its own tests
        e["SM_UMMA_FOLD"] = "0"
        e.update(env)
        p = subprocess.run([sys.executable, "-c", HASH_SNIPPET.format(root=ROOT)], env=e, capture_output=True,
                           text=True, timeout=600, cwd=ROOT)
        assert p.returncode == 0, p.stdout[-2000:] + p.stderr[-4000:]
        line = [ln for ln in p.stdout.splitlines() if ln.startswith("HASH")][0].split()
        seen[tuple(sorted(env.items()))] = (line[1], float(line[2]), float(line[3]))
    x_hashes = {v[0] for v in seen.values()}
    assert len(x_hashes) == 1, seen
    # residual partial sums are grouped per (tile, CTA, warp): the two tile geometries (128- and 256-row tiles) sum the
    # same fp32 squares in a different grouping, so the residuals agree to fp32 rounding, not to the bit
    ref = next(iter(seen.values()))
    for v in seen.values():
        assert abs(v[1] - ref[1]) <= 1e-6 * abs(ref[1]) and abs(v[2] - ref[2]) <= 1e-6 * abs(ref[2]), seen


def test_share_a_is_bit_identical_with_the_folded_geometry():
    """umma.sharea only changes where product 1 reads its A rows from (the B stage instead of a copy of their own) and
    which of a panel's tiles is the narrow one: every output element is the same k-ordered sum, so the iterates of the
    default (folded) geometry agree to the bit with and without it, per-phase launches and stream mode."""
    for base in ({"SM_UMMA_RESIDENT": "0"}, {"SM_UMMA_RESIDENT": "0", "SM_UMMA_STREAM": "1"}):
        hashes = []
        for v in ("0", "1"):
            e = dict(os.environ)
            e.update(base)
            e["SM_UMMA_SHAREA"] = v
            p = subprocess.run([sys.executable, "-c", HASH_SNIPPET.format(root=ROOT)], env=e, capture_output=True,
                               text=True, timeout=600, cwd=ROOT)
            assert p.returncode == 0, p.stdout[-2000:] + p.stderr[-4000:]
            hashes.append([ln for ln in p.stdout.splitlines() if ln.startswith("HASH")][0].split()[1])
        assert hashes[0] == hashes[1], (base, hashes)
