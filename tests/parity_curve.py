"""Per-chunk parity curve of a full-size config (not a pytest module; run by hand on a GPU box):

    python tests/parity_curve.py cfg5 2,5 [max_chunks] [field=value ...]     (e.g. l2_k=1 renorm=1)

streams the whole config through the CUDA path (all heads) and through the float64 oracle (the listed
heads: heads are independent, so this is exact per head) and prints, per chunk, the errors of O and of
the fast weights next to the oracle's own sensitivity: a second float64 run whose INITIAL weights
were rounded to bf16 once (the floor any bf16-operand implementation can be
asked to meet). Results of round 1 are in DESIGN.md section 7."""
import sys, os, time
sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
import numpy as np
import torch
import ttt_inputs as ti
from oracle.ttt_oracle import OracleTTT, rel_err
from paper_2604_08542_b200 import TTT, TTT_BF16

name = sys.argv[1]; heads = [int(x) for x in sys.argv[2].split(",")]
nmax = int(sys.argv[3]) if len(sys.argv) > 3 and "=" not in sys.argv[3] else 10**9
w = ti.CONFIGS[name]; dev = torch.device("cuda", 0)
over = {}
for a in sys.argv[3:]:
    if "=" in a:
        k, v = a.split("=")
        over[k] = type(getattr(w, k))(int(v)) if not isinstance(getattr(w, k), float) else float(v)
if over:
    w = ti.scaled(w, **over)
    print("# overrides:", over)
W1, W2, W3 = ti.fast_weights(w)
cols = torch.cat([torch.arange(h * w.hd, (h + 1) * w.hd) for h in heads])
r = lambda x: x.to(torch.bfloat16).to(torch.float32)
ora = OracleTTT(W1[heads], W2[heads], W3[heads], ns_iters=w.ns_iters, renorm=w.renorm)
flo = OracleTTT(r(W1[heads]), r(W2[heads]), r(W3[heads]), ns_iters=w.ns_iters, renorm=w.renorm)
gpu = TTT(w.nh, w.hd, w.hidden, TTT_BF16, ns_iters=w.ns_iters, renorm=w.renorm, max_tokens=w.chunk_tokens)
gpu.ttt_init(W1.to(dev), W2.to(dev), W3.to(dev))
out = sys.stdout
print("# chunk  err_O(gpu)  err_W(gpu)  floor_O  floor_W  rms(O_ref)  |W1|_F/head", file=out, flush=True)
t0 = time.time()
for c, (Q, K, V, lr) in enumerate(ti.TokenStream(w)):
    if c >= nmax: break
    O = gpu.ttt_chunk_step(Q.to(dev), K.to(dev), V.to(dev), lr.to(dev))
    a = (Q[:, cols].contiguous(), K[:, cols].contiguous(), V[:, cols].contiguous(), lr[heads].contiguous())
    O_ref, _ = ora.chunk_step(*a)
    O_flo, _ = flo.chunk_step(*a)
    g = [x.cpu()[heads] for x in gpu.ttt_get_weights()]
    ew = max(rel_err(g[0], ora.W1), rel_err(g[1], ora.W2), rel_err(g[2], ora.W3))
    fw = max(rel_err(flo.W1, ora.W1), rel_err(flo.W2, ora.W2), rel_err(flo.W3, ora.W3))
    print(c, "%.3e %.3e %.3e %.3e %.3e %.3e" % (rel_err(O[:, cols.to(dev)].float().cpu(), O_ref), ew,
          rel_err(O_flo, O_ref), fw, float(np.sqrt((np.asarray(O_ref) ** 2).mean())),
          float(np.linalg.norm(np.asarray(ora.W1)) / len(heads) ** 0.5)), "t=%.0fs" % (time.time() - t0), file=out, flush=True)
