// reg_classes.h -- the l-classes served by the register family (reg_kernel.cuh), split into groups = translation units.
// Canonical classes only: la >= lb, lc >= ld, (la,lb) >= (lc,ld); lb, ld <= 1; see DESIGN.md "Kernel families".
#pragma once
#define REG_GROUP0(X) X(0,0,0,0) X(1,0,0,0) X(1,0,1,0) X(1,1,0,0) X(1,1,1,0) X(2,0,0,0) X(2,0,1,0) X(3,0,0,0)
#define REG_GROUP1(X) X(2,0,1,1) X(2,0,2,0) X(2,1,0,0) X(3,0,1,0) X(4,0,0,0)
#define REG_GROUP2(X) X(2,1,1,0) X(3,1,0,0) X(4,0,1,0) X(4,1,0,0)
#define REG_GROUP3(X) X(1,1,1,1) X(3,0,2,0)
