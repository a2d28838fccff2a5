"""One window of the products workload, four gathers, each followed by a GraphSAGE-mean training
step (gg_sage_step): the command profiles/r01_e_consumer.md profiles."""
import sys
sys.path.insert(0, __import__('os').path.dirname(__import__('os').path.dirname(__import__('os').path.dirname(__import__('os').path.abspath(__file__)))))
import numpy as np, torch
from paper_2606_02916_b200 import inputs, epoch as ep, binding, build
build.build_library()
dev = torch.device("cuda", 0)
w = inputs.make_workload("products", device=dev)
g = ep.graph_from_workload(w, max_window=4)
feats = torch.empty(500000, w.dim, dtype=w.dtype, device=dev)
dims = [100, 16, 16, 47]
rng = np.random.default_rng(7)
p0 = [dict(W_self=(rng.uniform(-1, 1, (dims[l], dims[l + 1])) / np.sqrt(dims[l])).astype(np.float32),
           W_neigh=(rng.uniform(-1, 1, (dims[l], dims[l + 1])) / np.sqrt(dims[l])).astype(np.float32),
           b=np.zeros(dims[l + 1], np.float32)) for l in range(3)]
model = binding.Sage(p0, dev)
labels = torch.randint(0, 47, (1024,), dtype=torch.int32, device=dev)
g.window_stage(0, 0, w.batches[:4], w.fanouts)
for j in range(4):
    r = g.batch_gather(0, j, feats)
    model.step(r, labels, 0.003)
torch.cuda.synchronize()
print("loss", float(model.loss.cpu()[0]), [ (b["n_dst"], b["n_src"], b["n_edge"]) for b in r["blocks"]])
g.window_release(0); g.close()
