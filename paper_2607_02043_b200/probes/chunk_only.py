"""Chunk-only throughput of the pair kernel (no decodes): python -m paper_2607_02043_b200.probes.chunk_only (needs a B200)."""
import os, sys, time
sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__)))))
import numpy as np, torch
from paper_2607_02043_b200 import kairos as K, workloads as W
def ev(): return torch.cuda.Event(enable_timing=True)
def bench(C, P):
    inp = W.make_inputs("x", 5, [], C, P)
    pool = K.bf16_tensor(inp.pool); ws = torch.empty(K.workspace_bytes(1, C), dtype=torch.uint8, device="cuda")
    ctx = K.Kairos(pool, ws, inp.softmax_scale)
    cpt=torch.from_numpy(inp.chunk_page_table).cuda(); dpt=torch.zeros((1,1),dtype=torch.int32,device="cuda")
    qd=torch.empty((0,16,576),dtype=torch.bfloat16,device="cuda"); qc=K.bf16_tensor(inp.q_chunk)
    oc=torch.empty((C,16,512),dtype=torch.bfloat16,device="cuda"); od=torch.empty((0,16,512),dtype=torch.bfloat16,device="cuda")
    f=lambda: ctx.mixed_step(qd, dpt, np.zeros(0,np.int32), qc, cpt, C, P, out_dec=od, out_chunk=oc, want_lse=False)
    for _ in range(3): f()
    torch.cuda.synchronize(); e0,e1=ev(),ev(); e0.record()
    n=10
    for _ in range(n): f()
    e1.record(); torch.cuda.synchronize()
    us=e0.elapsed_time(e1)*1e3/n
    tiles=(C+7)//8; pp=sum(-(-(P+min(C,(t+1)*8))//64) for t in range(tiles))
    info=ctx.last_plan_info()
    npair=min(74,tiles)
    flops=34816*(C*P+C*(C+1)//2)
    print(f"C={C} P={P}: {us:8.1f} us  pair-pages={pp} tiles={tiles} -> {us*1.965e3*npair/pp:7.0f} cycles/pair-page (if {npair} pairs)  {flops/us/1e6:7.1f} TFLOP/s  kernels={info['kernels']}")
for C,P in [(8192,0),(4096,0),(2048,6144),(2048,0),(1024,0),(4096,28672),(592,20000)]:
    bench(C,P)
