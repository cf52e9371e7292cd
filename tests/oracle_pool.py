"""Fan independent CPU-oracle calls out over worker processes (test infrastructure).

The oracle is single-threaded; SURVEY.md 8(d) allows the harness to run independent rotations / output ciphertexts in P
worker processes of the same single-threaded program.  Workers are forked, so they see the parent's oracle objects
(parameters, keys, ciphertexts) without pickling them; only the small job tuples go in and numpy arrays come back.
Workers never touch CUDA."""
import multiprocessing as mp
import os

import numpy as np

_SHARED = None


def _work(job):
    fn, args = job
    return fn(_SHARED, *args)


def pmap(shared, fn, arglist, procs=None):
    """[fn(shared, *args) for args in arglist], in forked worker processes when there is more than one job."""
    global _SHARED
    arglist = list(arglist)
    procs = procs or min(len(arglist), os.cpu_count() or 1, 24)
    if procs <= 1 or len(arglist) <= 1:
        return [fn(shared, *a) for a in arglist]
    _SHARED = shared
    try:
        with mp.get_context("fork").Pool(procs) as pool:
            # a bounded wait: a worker that deadlocked in fork() must fail the test, not hang the box
            return pool.map_async(_work, [(fn, a) for a in arglist], chunksize=1).get(timeout=2400)
    finally:
        _SHARED = None


# ---- jobs (shared = dict with ck, P, keys and whatever the job reads)
def job_rotate(sh, src_key, amt, hoisted):
    ck = sh["ck"]
    f = ck.rotate_hoisted if hoisted else ck.rotate
    return f(sh["P"], sh["keys"], sh["inputs"][src_key], amt).c


def job_mac(sh, terms):
    """sum of ct (*) pt over terms [(ct_key, pt_key)]; ct_key indexes sh['cts'], pt_key sh['pts'] -> [2][L][N]"""
    ck, P = sh["ck"], sh["P"]
    first = sh["cts"][terms[0][0]]
    acc = np.zeros_like(first.c)
    for ck_, pk in terms:
        ck.pmult_acc(P, acc, sh["cts"][ck_], sh["pts"][pk])
    return acc


def job_rotate_ct(sh, idx, amt):
    return sh["ck"].rotate(sh["P"], sh["keys"], sh["outer"][idx], amt).c
