"""Self-check of an installed libgs on the current GPU: every compute entry point of include/gs.h once, at small
ragged sizes, real and complex, verified by the defining identities of PAPER.md:63-67 (U^H U = S, U U^-1 = I,
U^H H~ U = H, U C = C~) evaluated with plain torch -- no oracle, no reference library.

    python -m paper_2502_02460_b200.selfcheck [--sizes 100 257] [--standard-evp]

It is also the program the memory / race checkers are pointed at (profiles/r02_sanitizer.md):

    compute-sanitizer --tool memcheck  python -m paper_2502_02460_b200.selfcheck
    compute-sanitizer --tool racecheck python -m paper_2502_02460_b200.selfcheck
"""
from __future__ import annotations

import argparse
import sys

import torch

from . import gs, sharded
from . import workloads as wl


def _rel(a: torch.Tensor, b: torch.Tensor) -> float:
    return ((a - b).norm() / b.norm().clamp_min(1e-300)).item()


def check_size(N: int, cplx: bool, standard_evp: bool = False) -> dict:
    dt = torch.complex128 if cplx else torch.float64
    nev = max(1, (2 * N) // 3)
    p = wl.small_pencil(N, seed=N, complex=cplx, device="cuda")
    plan, U, V, Ht = gs.generalized_to_standard(p.H, p.S, nev)
    out = {}
    Ut = torch.triu(U)
    out["chol"] = _rel(Ut.conj().t() @ Ut, p.S)
    out["inv"] = ((Ut @ V - torch.eye(N, dtype=dt, device="cuda")).norm() / N ** 0.5).item()
    Hs = torch.triu(Ht) + torch.triu(Ht, 1).conj().t()
    out["std"] = _rel(Ut.conj().t() @ (Hs @ Ut), p.H)
    Ct = wl.dense_rhs(N, nev, seed=1, complex=cplx, device="cuda")
    C = wl.colmajor_empty(N, nev, dtype=dt, device="cuda")
    plan.backtransform(V, Ct, C)
    plan.last_info()
    out["back"] = _rel(Ut @ C, Ct)
    f = torch.linspace(2.0, 0.0, nev, dtype=torch.float64, device="cuda")
    P = wl.colmajor_zeros(N, N, dtype=dt, device="cuda")
    plan.density_matrix(C, f, P)
    plan.last_info()
    Pref = (C.conj() * f.to(dt)) @ C.t()
    out["dens"] = _rel(torch.triu(P), torch.triu(Pref))
    # column-range (sharded) forms: two ranges, the second buffer as push target
    Vx, Gx, Htx, Vw, Ux = (wl.colmajor_zeros(N, N, dtype=dt, device="cuda") for _ in range(5))
    plan.set_push_targets(gs.GS_PUSH_UINV, [Vx.data_ptr()])
    ranges = sharded.column_ranges(N, 2, plan.block)
    for c0, c1 in ranges:
        if c1 > c0:
            Ux.copy_(p.S)
            plan.cholesky_leading(Ux, c1)
            plan.invert_triangular_cols(Ux, Vw, c0, c1 - c0)
            plan.to_standard_g_cols(p.H, Vw, Gx, c0, c1 - c0)
    for c0, c1 in ranges:
        if c1 > c0:
            plan.to_standard_cols(Vx, Gx, Htx, c0, c1 - c0)
    plan.backtransform_cols(V, Ct, C, 0, nev)
    plan.last_info()
    plan.set_push_targets(gs.GS_PUSH_UINV, [])
    out["cols_inv"] = _rel(torch.triu(Vx), torch.triu(V))
    out["cols_std"] = _rel(torch.triu(Htx), torch.triu(Ht))
    # step 1 in its sharded form (one rank: no peers) and the allocation-free density matrix
    Us = wl.colmajor_empty(N, N, dtype=dt, device="cuda")
    Us.copy_(p.S)
    plan.cholesky_sharded(Us, 0, 1)
    Ps = wl.colmajor_zeros(N, N, dtype=dt, device="cuda")
    plan.density_matrix_static(C, f, Ps)
    plan.last_info()
    Ust = torch.triu(Us)
    out["chol_sharded"] = _rel(Ust.conj().t() @ Ust, p.S)
    out["dens_static"] = _rel(torch.triu(Ps), torch.triu(Pref))
    if standard_evp and hasattr(plan, "standard_eigh"):
        eps, Q = plan.standard_eigh(Ht.clone())
        plan.last_info()
        R = Hs @ Q - Q * eps.to(dt).unsqueeze(0)
        out["evp_resid"] = (R.norm() / (Hs.norm() * N * 2.0 ** -52)).item()
        G = Q.conj().t() @ Q
        G.diagonal().sub_(1.0)
        out["evp_orth"] = G.abs().max().item()
        lam = plan.standard_eigenvalues(Ht.clone(), count=eps.numel())   # eigenvalues only: bisection instead of Solve and Back
        plan.last_info()
        out["evp_bisect"] = ((lam - eps).abs().max() / max(1.0, eps.abs().max().item())).item()
        # the whole generalized solve in one call: H C = S C eps, C^H S C = I
        eps_g, Cg, _, _ = plan.generalized_eigh(p.H, p.S)
        plan.last_info()
        Rg = p.H @ Cg - (p.S @ Cg) * eps_g.to(dt).unsqueeze(0)
        out["gen_resid"] = (Rg.norm() / (p.H.norm() * N * 2.0 ** -52)).item()
        Gg = Cg.conj().t() @ (p.S @ Cg)
        Gg.diagonal().sub_(1.0)
        out["gen_sorth"] = Gg.abs().max().item()
    plan.close()
    return out


def main(argv=None) -> int:
    ap = argparse.ArgumentParser()
    ap.add_argument("--sizes", type=int, nargs="*", default=[100, 257])
    ap.add_argument("--standard-evp", action="store_true", help="also run the standard eigensolver (NEXT-4)")
    args = ap.parse_args(argv)
    if not torch.cuda.is_available():
        print("selfcheck: no CUDA device (libgs has no CPU fallback)", file=sys.stderr)
        return 2
    bad = 0
    for N in args.sizes:
        for cplx in (False, True):
            r = check_size(N, cplx, args.standard_evp)
            tol = {"chol": 1e-13, "inv": 1e-11, "std": 1e-9, "back": 1e-11, "dens": 1e-12, "cols_inv": 1e-11, "cols_std": 1e-11,
                   "evp_resid": 100.0, "evp_orth": 1e-11, "chol_sharded": 1e-13, "dens_static": 1e-12, "gen_resid": 100.0, "gen_sorth": 1e-10, "evp_bisect": 1e-12}
            ok = all(v <= tol[k] for k, v in r.items())
            bad += 0 if ok else 1
            print(f"selfcheck N={N} {'c128' if cplx else 'f64'} {'ok' if ok else 'FAILED'} " +
                  " ".join(f"{k}={v:.2e}" for k, v in r.items()))
    torch.cuda.synchronize()
    return 1 if bad else 0


if __name__ == "__main__":
    sys.exit(main())
