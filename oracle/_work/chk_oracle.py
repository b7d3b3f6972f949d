import numpy as np, sys, time
sys.path.insert(0, '/root/repo')
from oracle import *
A = np.array([[1.,2],[3,4]])
for nf, exp in ((2,(2,32,-48)),(3,(6,96,-720))):
    print('TV1', nf, o1_all_subsets(A[None], nf, None, sb=False), o3_uniform(A, nf, 0.0, True), exp)
A2 = np.array([[2.,-1,3],[1,4,-2],[-3,5,1]])
print('TV2', o1_all_subsets(A2[None], 2, None, sb=False), o3_uniform(A2,2,0.0,True), o2a_twospin(A2,A2))
print('TV2 nf3', o1_all_subsets(A2[None], 3, None, sb=False), o3_uniform(A2,3,0.0,True))
A0=np.array([[1.,2],[3,4]]); A1=np.array([[2.,-1],[1,3]]); Ab=np.stack([A0,A1]); sg=[0.5,-1/3]
print('TV3', o1_all_subsets(Ab,2,sg,sb=True), o2b_polynomial(Ab,sg), o2a_twospin(A0,A1,sg[0],sg[1]), [11/3,26,-2018/9])
print('TV3 alg3 full', o3_alg3(Ab,sg), 'single0', o3_alg3(Ab[:,:1,:1],sg))
A2_=np.array([[-1.,1],[2,1]]); Ac=np.stack([A0,A1,A2_]); sg3=[0.5,0,-0.5]
print('TV4', o1_all_subsets(Ac,3,sg3,sb=True), o2b_polynomial(Ac,sg3), o3_alg3(Ac,sg3))
rng=np.random.default_rng(5)
for n in (2,3,4):
  for nf in (2,3):
    A=rng.standard_normal((nf,n,n)); sg=rng.standard_normal(nf)
    t=time.time(); a=o1_connected(A,nf,sg,True); t1=time.time()-t
    b=o3_alg3(A,sg); c=o2b_polynomial(A,sg)[-1]
    print(n,nf,a,b,c,'t',t1)
    Au=A[:1]; s0=sg[0]
    a=o1_connected(Au,nf,[s0],False); b=o3_uniform(Au[0],nf,s0,False)[0]
    e=o1_connected(np.repeat(Au,nf,0),nf,[s0]*nf,True)
    print('  uni',a,b,'sb-equal',e)
    print('  abs', o1_connected(A,nf,sg,True,True), o3_alg3(A,sg,True), o1_connected(Au,nf,None,False,True), o3_uniform(Au[0],nf,0,False,True)[0])
